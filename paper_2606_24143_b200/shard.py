"""Host logic of the token-sharded (data-parallel) use of the OPD loss: one process per GPU, every rank holds all
of W and a contiguous range of whole sequences (rows are independent given W).  No collective sits on
the data path of the loss itself; a trainer needs exactly three small exchanges around it:

    N_global = all_reduce(sum)(N_local)           before the call -> pass norm_override = N_global
    loss     = all_reduce(sum)(loss_local)        (each local loss is already divided by N_global)
    grad_W   = all_reduce(sum)(grad_W_local)      fp32 d x V (2.49 GB at C4; NCCL over NVLink/NVSwitch)

grad_hidden stays local.  `engine` is any callable with the opd_loss_fwd_bwd signature returning a dict with
loss / grad_W tensors (the CUDA binding in production; the tests drive this module with the CPU oracle over gloo).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def token_shard(seq_lens, rank: int, world: int):
    """Split whole sequences over ranks, balancing tokens greedily in order. Returns (first_token, last_token_excl)."""
    total = int(sum(seq_lens))
    bounds = [0]
    acc = 0
    target = total / world
    r = 1
    for n in seq_lens:
        acc += int(n)
        while r < world and acc >= target * r - 1e-9:
            bounds.append(acc)
            r += 1
    while len(bounds) < world:
        bounds.append(total)
    bounds.append(total)
    return bounds[rank], bounds[rank + 1]


def global_live_count(mask_local: torch.Tensor, group=None) -> float:
    n = torch.tensor([float((mask_local != 0).sum().item())], dtype=torch.float64, device=mask_local.device)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(n, group=group)
    return float(n.item())


def sharded_loss_fwd_bwd(engine, hidden, W, cache_idx, lam, old, mask, mode, k_or_K, group=None, **kw):
    """Run `engine` on this rank's token shard with the global normaliser and combine loss and grad_W over ranks."""
    n_global = global_live_count(mask, group)
    out = engine(hidden, W, cache_idx, lam, old, mask, mode, k_or_K, norm_override=n_global if n_global > 0 else 0.0, **kw)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(out["loss"], group=group)
        if out.get("grad_W") is not None:
            dist.all_reduce(out["grad_W"], group=group)
    out["N_global"] = n_global
    return out

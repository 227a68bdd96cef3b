"""Seeded synthetic workloads for the fused OPD loss (shared by tests, bench.py and the oracle tests).

This module only *generates inputs*: student hidden states and head, an independent teacher
head, a stale ("old") student head, and the finite caches the learner receives
(cached actions, teacher scores on them, rollout-time log-probs).  It holds
none of the loss / estimator arithmetic and imports neither the CUDA binding nor the oracle.

Recipe (shapes from BASELINE.json configs):
  seeds          s(c, i) = 20260624 + 1000*c + i   for config c, stream i
  hidden         ~ N(0,1)                          (i=0)
  W32            ~ N(0,1/d), W = cast(W32)         (i=1)       logical [d,V], v contiguous
  teacher W_T    ~ N(0,1/d) independent            (i=2)       log q = logsoftmax(hidden @ W_T), temperature 1
  stale student  W_old = cast(W32 + sigma*E), E ~ N(0,1/d) (i=3); sigma=0 => W_old == W bit for bit
  mask           (i=4)   'none' | 'random10' (exactly floor(0.1*T) masked) | 'varlen' (sequences padded
                         to seq_len, lengths uniform in [min_len, seq_len], i=6)
  MC draws       (i=5)   a_j ~ Categorical(p_old) iid WITH replacement, K per token
  top-k cache    idx = TopK(log q, k) chosen by the teacher, lam = log q[idx]
  MC cache       idx = a, lam = log q[a], old = log p_old[a]
  stale top-k    idx = TopK(log p_old, k) (the rollout-time student support S_old), lam = log q[idx]
Stress variants (reported / tested, not bench configs): cfg["hidden_scale"] = 4 gives PEAKED rows (logits of
standard deviation 4: a few columns hold most of the mass, most exponentials are tiny); cfg["order"] = "monotone" scales
column v of the student heads by 0.5 + 1.5 v/V, so column norms grow with the index and the running maximum of a row keeps
moving to later vocabulary tiles (online-max rescaling); a large sigma gives heavy importance-ratio tails.
cfg["hot_columns"] = h gives SKEWED SUPPORTS: h fixed columns (spread over the vocabulary: v_i = (i * 9973 + 7) mod V) are
put into the last h slots of every row's top-k caches (teacher's and stale student's) unless the row already holds them, with
the teacher's log-prob of that column; real LM supports look like this (a few very common tokens sit in most rows' top-k), and
one column then owns about T of the T*k cache entries.  Indices stay distinct within a row.
All cache values are fp32, indices int32.  Rollout settings follow PAPER.md:332 (temperature 1,
no truncation).  These are stand-ins for the paper's Qwen3 workloads: V=151936 and
d in {2048,2560,4096} are the 1.7B/4B/8B-class student heads.
"""
from __future__ import annotations

import torch

SEED0 = 20260624

# BASELINE.json configs (index = position in BASELINE.json "configs", 1-based to match DESIGN.md C1..C5)
CONFIGS = {
    1: dict(name="C1", dtype="fp32", T=256, d=256, V=4096, k=8, K=4, sigma=0.05, mask="random10"),
    2: dict(name="C2", dtype="bf16", T=4096, d=1024, V=32768, k=16, K=4, sigma=0.02, mask="none"),
    3: dict(name="C3", dtype="bf16", T=16384, d=2048, V=151936, k=32, K=8, sigma=0.02, mask="varlen",
            seq_len=4096, min_len=512),
    4: dict(name="C4", dtype="bf16", T=32768, d=4096, V=151936, k=16, K=16, sigma=0.02, mask="none"),
    5: dict(name="C5", dtype="bf16", T=65536, d=2560, V=151936, k=64, K=8, sigma=0.02, mask="mixed_seq",
            seq_len=8192),
}


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def _tdtype(name: str):
    return torch.bfloat16 if name == "bf16" else torch.float32


def make_mask(cfg: dict, c: int, device="cpu") -> torch.Tensor:
    """uint8 [T]; 0 = masked, 1 = live (in 'mixed_seq': 1 = FKL_TOPK row, 2 = RKL_MC row)."""
    T = cfg["T"]
    kind = cfg.get("mask", "none")
    if kind == "none":
        return torch.ones(T, dtype=torch.uint8, device=device)
    if kind == "random10":
        g = _gen(SEED0 + 1000 * c + 4, "cpu")
        perm = torch.randperm(T, generator=g)
        m = torch.ones(T, dtype=torch.uint8)
        m[perm[: T // 10]] = 0
        return m.to(device)
    if kind == "varlen":
        L = cfg["seq_len"]
        nseq = T // L
        g = _gen(SEED0 + 1000 * c + 6, "cpu")
        lens = torch.randint(cfg["min_len"], L + 1, (nseq,), generator=g)
        pos = torch.arange(L).unsqueeze(0).expand(nseq, L)
        return (pos < lens.unsqueeze(1)).to(torch.uint8).reshape(T).to(device)
    if kind == "mixed_seq":
        L = cfg["seq_len"]
        nseq = T // L
        code = torch.ones(nseq, dtype=torch.uint8)
        code[nseq // 2:] = 2          # first half of the sequences FKL_TOPK, second half RKL_MC
        return code.repeat_interleave(L).to(device)
    raise ValueError(kind)


def make_inputs(cfg: dict, c: int = 0, device="cpu", keep_teacher_rows: bool = False,
                chunk: int = 2048, sigma=None) -> dict:
    """Generate one workload.  Returns tensors on ``device``:

    hidden [T,d], W [d,V] (cfg dtype); mask [T] u8;
    topk_idx [T,k] i32, topk_logq [T,k] f32            (teacher-selected support + its log-probs)
    mc_idx [T,K] i32, mc_logq [T,K] f32, mc_logp_old [T,K] f32
    stopk_idx [T,k] i32, stopk_logq [T,k] f32         (stale student's top-k support S_old + teacher log-probs on it)
    and, if keep_teacher_rows, logq [T,V] / logp_old [T,V] f32 (small configs, for oracle pins).
    """
    T, d, V, k, K = cfg["T"], cfg["d"], cfg["V"], cfg["k"], cfg["K"]
    sig = cfg["sigma"] if sigma is None else sigma
    dt = _tdtype(cfg["dtype"])
    dev = torch.device(device)
    s = SEED0 + 1000 * c
    hidden = (torch.randn(T, d, generator=_gen(s + 0, dev), device=dev, dtype=torch.float32) * float(cfg.get("hidden_scale", 1.0))).to(dt)
    W32 = torch.randn(d, V, generator=_gen(s + 1, dev), device=dev, dtype=torch.float32) * (d ** -0.5)
    ramp = None
    if cfg.get("order") == "monotone":
        ramp = 0.5 + 1.5 * torch.arange(V, device=dev, dtype=torch.float32) / V
        W32 = W32 * ramp
    W = W32.to(dt)
    WT = (torch.randn(d, V, generator=_gen(s + 2, dev), device=dev, dtype=torch.float32) * (d ** -0.5)).to(dt)
    if sig == 0:
        Wold = W
    else:
        E = torch.randn(d, V, generator=_gen(s + 3, dev), device=dev, dtype=torch.float32) * (d ** -0.5)
        if ramp is not None:
            E = E * ramp
        Wold = (W32 + sig * E).to(dt)
        del E
    del W32
    g5 = _gen(s + 5, dev)

    topk_idx = torch.empty(T, k, dtype=torch.int32, device=dev)
    topk_logq = torch.empty(T, k, dtype=torch.float32, device=dev)
    stopk_idx = torch.empty(T, k, dtype=torch.int32, device=dev)
    stopk_logq = torch.empty(T, k, dtype=torch.float32, device=dev)
    mc_idx = torch.empty(T, K, dtype=torch.int32, device=dev)
    mc_logq = torch.empty(T, K, dtype=torch.float32, device=dev)
    mc_old = torch.empty(T, K, dtype=torch.float32, device=dev)
    logq_all = torch.empty(T, V, dtype=torch.float32, device=dev) if keep_teacher_rows else None
    logpold_all = torch.empty(T, V, dtype=torch.float32, device=dev) if keep_teacher_rows else None
    WTf, Woldf = WT.float(), Wold.float()
    for r0 in range(0, T, chunk):
        r1 = min(T, r0 + chunk)
        h = hidden[r0:r1].float()
        logq = torch.log_softmax(h @ WTf, dim=-1)
        logpo = torch.log_softmax(h @ Woldf, dim=-1)
        tv, ti = torch.topk(logq, k, dim=-1)               # descending
        si = torch.topk(logpo, k, dim=-1).indices            # stale student's support S_old = TopK(p_old, k)
        for j in range(int(cfg.get("hot_columns", 0))):      # skewed supports: see the module docstring
            col = (j * 9973 + 7) % V
            for sup in (ti, si):
                sup[~(sup == col).any(dim=1), k - 1 - j] = col
        if cfg.get("hot_columns"):
            tv = torch.gather(logq, 1, ti)
        topk_idx[r0:r1] = ti.to(torch.int32)
        topk_logq[r0:r1] = tv
        stopk_idx[r0:r1] = si.to(torch.int32)
        stopk_logq[r0:r1] = torch.gather(logq, 1, si)
        a = torch.multinomial(torch.exp(logpo), K, replacement=True, generator=g5)
        mc_idx[r0:r1] = a.to(torch.int32)
        mc_logq[r0:r1] = torch.gather(logq, 1, a)
        mc_old[r0:r1] = torch.gather(logpo, 1, a)
        if keep_teacher_rows:
            logq_all[r0:r1] = logq
            logpold_all[r0:r1] = logpo
    out = dict(hidden=hidden, W=W, mask=make_mask(cfg, c, dev), topk_idx=topk_idx, topk_logq=topk_logq,
               mc_idx=mc_idx, mc_logq=mc_logq, mc_logp_old=mc_old, stopk_idx=stopk_idx, stopk_logq=stopk_logq,
               cfg=dict(cfg), sigma=sig)
    if keep_teacher_rows:
        out["logq"] = logq_all
        out["logp_old"] = logpold_all
        out["W_old"] = Wold
        out["W_T"] = WT
    return out


def mixed_cache(inp: dict):
    """One [T,C] cache for OPD_MIXED, C = max(k,K): FKL rows (mask==1) hold the top-k cache in their
    first k slots, MC rows (mask==2) the MC cache in their first K slots; unused slots are zero."""
    k = inp["topk_idx"].shape[1]
    K = inp["mc_idx"].shape[1]
    C = max(k, K)
    T = inp["mask"].shape[0]
    dev = inp["mask"].device
    idx = torch.zeros(T, C, dtype=torch.int32, device=dev)
    lam = torch.zeros(T, C, dtype=torch.float32, device=dev)
    old = torch.zeros(T, C, dtype=torch.float32, device=dev)
    f = inp["mask"] == 1
    m = inp["mask"] == 2
    idx[f, :k] = inp["topk_idx"][f]
    lam[f, :k] = inp["topk_logq"][f]
    idx[m, :K] = inp["mc_idx"][m]
    lam[m, :K] = inp["mc_logq"][m]
    old[m, :K] = inp["mc_logp_old"][m]
    return idx, lam, old, k | (K << 16)

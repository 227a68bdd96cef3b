"""fp64 CPU oracle for the fused OPD loss (AsyncOPD, arxiv/paper_2606_24143).

TEST INFRASTRUCTURE ONLY.  Nothing on the product path may import this module:
only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs call it.  It shares no code with the CUDA path
(``paper_2606_24143_b200/``) and imports nothing from it.

What it computes, in the paper's order and notation (PAPER.md = /root/reference/PAPER.md):

  O1  z_t = x_t . W                      student logits over the whole vocabulary
                                         (p_theta(.|s) is a policy over V)
  O2  lse_t = log sum_v exp z_tv         two-pass stable softmax; logp = z - lse
  O3  l_tj = logp_t[a_tj]                current-student log-prob at the cached actions
                                         ("recompute log p_theta(a|s) for a in C_score(s)")
  O4  FKL_TOPK (Eq.(1) restricted to the cached support S, PAPER.md:74;
      renormalisers Z_q^S, Z_p^S of Eq.(9))
          logZq = log sum_j exp lam_j   (0 with NO_RENORM_TEACHER)
          logZp = log sum_j exp l_j     (only with RENORM_STUDENT, else 0)
          q~_j  = exp(lam_j - logZq)
          L_t   = sum_j q~_j [ (lam_j - logZq) - (l_j - logZp) ]
  O5  RKL_MC (PAPER.md:191 and Eq.(15); duplicates allowed)
          A_j   = lam_j - l_j                 (A_theta recomputed at learner time)
          rho_j = exp(l_j - o_j)              (unclipped old->current ratio)
          L_t   = -(1/m) sum_j rho_j A_j
  O5b RKL_TOPK (App. A.1 Eq.(8)-(10); the cached support S is fixed)
          p~_j = exp(l_j - log sum_S exp l),  q~_j = exp(lam_j - log sum_S exp lam)
          L_t  = sum_j p~_j (log p~_j - log q~_j);   g = sum_j p~_j (log p~_j - log q~_j - L_t) e_{a_j}
  O6  N = sum_t [mask_t != 0] (or norm_override), loss = (1/N) sum_t L_t, per_token_kl = L_t (0 if masked)
  O7  g_tv = dL_t/dz_tv with A frozen (stop-gradient):
          FKL:                g = (sum_j q~_j) p - sum_j q~_j e_{a_j}
          FKL RENORM_STUDENT: g = sum_j (p~_j - q~_j) e_{a_j},  p~_j = exp(l_j - logZp)
          MC:                 g = c p - (1/m) sum_j rho_j A_j e_{a_j},   c = (1/m) sum_j rho_j A_j
  O8  grad_hidden[t,:] = (1/N) W g_t
  O9  grad_W          = (1/N) sum_t x_t g_t^T
  O10 dense references (pins only): D_F (Eq.(1)), D_R (Eq.(2))

Readings of the paper where it is silent or ambiguous are listed in DESIGN.md ("Readings").
Pins (tests/test_oracle_pins.py): k=V equals dense D_F; k=1 equals library cross-entropy; K=V uniform
proposal equals dense D_R; Eq.(5) by enumeration; on-policy unbiasedness; 1/m variance law; KL >= 0;
zero cases; central finite differences; softmax-shift invariance; mask/permutation invariance;
duplicates; the four PPO-style surrogates against Eq.(4)/(6)/(7) written out; the sequence-level diagnostics by
enumeration.  No function here is "parity unpinned".

Everything is float64.  A library matmul (numpy) serves as the O1 step; tokens are processed in
row chunks only to bound memory (rows are independent).  ``opd_oracle_loops`` is the same
mathematics as pure Python loops, for brute-force cross-checks on tiny shapes.
"""
from __future__ import annotations

import math

import numpy as np

# modes / flags: numeric values are part of the paper-facing interface in include/opd.h;
# they are restated here by hand (the oracle includes no product header).
FKL_TOPK = 0
RKL_MC = 1
MIXED = 2
RKL_TOPK = 3          # sparse top-k reverse KL on the cached support, App. A.1 Eq.(8)-(10)

F_NO_RENORM_TEACHER = 1
F_RENORM_STUDENT = 2

# surrogate variants of the 2x2 ablation (Eq.(6),(7)); THETA_NOCLIP is Eq.(15)
SUR_THETA_NOCLIP = 0
SUR_THETA_CLIP = 1
SUR_OLD_NOCLIP = 2
SUR_OLD_CLIP = 3


def logsumexp(v: np.ndarray) -> float:
    """log sum exp, two-pass (max first)."""
    v = np.asarray(v, dtype=np.float64)
    if v.size == 0:
        return -math.inf
    m = float(np.max(v))
    if not math.isfinite(m):
        return m
    return m + math.log(float(np.sum(np.exp(v - m))))


def log_softmax_rows(z: np.ndarray):
    """O2: returns (logp[T,V], lse[T])."""
    z = np.asarray(z, dtype=np.float64)
    m = np.max(z, axis=1, keepdims=True)
    lse = m[:, 0] + np.log(np.sum(np.exp(z - m), axis=1))
    return z - lse[:, None], lse


def dense_forward_kl(logq: np.ndarray, logp: np.ndarray) -> np.ndarray:
    """O10 / Eq.(1): D_F = sum_a q (log q - log p), per row."""
    q = np.exp(logq)
    return np.sum(q * (logq - logp), axis=-1)


def dense_reverse_kl(logq: np.ndarray, logp: np.ndarray) -> np.ndarray:
    """O10 / Eq.(2): D_R = - sum_a p (log q - log p), per row."""
    p = np.exp(logp)
    return -np.sum(p * (logq - logp), axis=-1)


def token_terms(mode: int, lam: np.ndarray, old, ell: np.ndarray, flags: int,
                surrogate: int = SUR_THETA_NOCLIP, clip_eps: float = 0.2):
    """O4/O5/O7 for ONE token.

    lam, old, ell: the C cached teacher log-probs, old-student log-probs, current-student log-probs.
    Returns (L_t, alpha, beta[C]) with  dL_t/dz_v = alpha * p_v + sum_j beta_j [a_j == v].
    """
    lam = np.asarray(lam, dtype=np.float64)
    ell = np.asarray(ell, dtype=np.float64)
    C = lam.shape[0]
    if mode == FKL_TOPK:
        logZq = 0.0 if (flags & F_NO_RENORM_TEACHER) else logsumexp(lam)
        qt = np.exp(lam - logZq)
        if flags & F_RENORM_STUDENT:
            logZp = logsumexp(ell)
            pt = np.exp(ell - logZp)
            L = float(np.sum(qt * ((lam - logZq) - (ell - logZp))))
            # d/dz of -sum_j q~_j (l_j - logZp) restricted to S: sum_j q~_j * p~ - q~  (p~ sums to 1)
            alpha = 0.0
            beta = float(np.sum(qt)) * pt - qt
        else:
            L = float(np.sum(qt * ((lam - logZq) - ell)))
            alpha = float(np.sum(qt))
            beta = -qt
        return L, alpha, beta
    if mode == RKL_MC:
        old = np.asarray(old, dtype=np.float64)
        m = C
        rho = np.exp(ell - old)
        if surrogate in (SUR_THETA_NOCLIP, SUR_THETA_CLIP):
            A = lam - ell                      # A_theta
        else:
            A = lam - old                      # A_old,
        if surrogate in (SUR_THETA_NOCLIP, SUR_OLD_NOCLIP):
            term = rho * A                     # Eq.(6)/(7) noclip, Eq.(15)
            w = rho * A                        # d term / d l_j  (A frozen, d rho = rho d l)
        else:
            rbar = np.clip(rho, 1.0 - clip_eps, 1.0 + clip_eps)
            unc = rho * A
            cl = rbar * A
            term = np.minimum(unc, cl)         # Eq.(4): min(rho A, clip(rho) A)
            # the gradient flows through rho only where the unclipped branch is the active minimum
            # (ties: unclipped branch), or where the clip is inactive (rbar == rho)
            active = (unc <= cl) | (rbar == rho)
            w = np.where(active, rho * A, 0.0)
        L = -float(np.sum(term)) / m
        c = float(np.sum(w)) / m
        alpha = c
        beta = -w / m
        return L, alpha, beta
    if mode == RKL_TOPK:
        # Eq.(10) on the cached support, both distributions renormalised on S (Eq.(9)); the support is fixed during
        # the update, so dD/dz_v = sum_j dD/dl_j [a_j = v] and the full-vocabulary lse cancels.
        D, dD = sparse_reverse_kl(lam, ell)
        return D, 0.0, dD
    raise ValueError("mode must be FKL_TOPK, RKL_MC or RKL_TOPK per token")


def _split_k(mode: int, k_or_K: int):
    if mode == MIXED:
        return k_or_K & 0xFFFF, (k_or_K >> 16) & 0xFFFF
    return k_or_K, k_or_K


def opd_oracle(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K,
               flags: int = 0, norm_override: float = 0.0, want_grads: bool = True,
               want_grad_W: bool = True, rows=None, chunk: int = 512,
               surrogate: int = SUR_THETA_NOCLIP, clip_eps: float = 0.2):
    """The whole path O1-O9 in float64.

    hidden [T,d]; W logical [d,V] (any strides: pass a transposed view for a [V,d] weight);
    cache_idx [T,C] ints in [0,V); cache_teacher_logp / cache_old_logp [T,C]; mask [T]
    (0 = masked; in MIXED 1 = FKL_TOPK row, 2 = RKL_MC row).  FKL rows use the first k cache
    slots, MC rows the first K.  ``rows``: optional list of token indices — only those rows are
    evaluated (N is still the full live count) and grad_W is then the partial sum over them.

    Returns dict: loss, N, per_token_kl[T], lse[T], student_logp[T,C] (NaN in unused slots),
    alpha[T], grad_hidden[T,d], grad_W[d,V].
    """
    X = np.asarray(hidden, dtype=np.float64)
    Wd = np.asarray(W, dtype=np.float64)
    idx = np.asarray(cache_idx).astype(np.int64)
    lam_all = np.asarray(cache_teacher_logp, dtype=np.float64)
    old_all = None if cache_old_logp is None else np.asarray(cache_old_logp, dtype=np.float64)
    msk = np.asarray(mask).astype(np.int64)
    T, d = X.shape
    V = Wd.shape[1]
    assert Wd.shape[0] == d
    k_f, K_m = _split_k(mode, k_or_K)

    N = float(np.count_nonzero(msk))
    norm = float(norm_override) if norm_override > 0 else N
    scale = 0.0 if norm == 0 else 1.0 / norm

    per_token = np.zeros(T)
    lse_out = np.zeros(T)
    alpha_out = np.zeros(T)
    slp = np.full(idx.shape, np.nan)
    rho_out = np.full(idx.shape, np.nan)       # diagnostics: rho_theta(a_tj) on MC rows (Fig. 5)
    var1_out = np.zeros(T)                     # diagnostics: sample variance of the one-sample terms (Eq.(16))
    first_out = np.zeros(T)                    # diagnostics: L^MC_1 from the first cached draw, -rho_1 A_theta,1 (Eq.(15), m = 1)
    gh = np.zeros((T, d)) if want_grads else None
    gW = np.zeros((d, V)) if (want_grads and want_grad_W) else None

    live = np.flatnonzero(msk) if rows is None else np.asarray([r for r in rows if msk[r] != 0], dtype=np.int64)
    for s in range(0, live.size, chunk):
        tt = live[s:s + chunk]
        z = X[tt] @ Wd                                     # O1
        logp, lse = log_softmax_rows(z)                    # O2
        p = np.exp(logp) if want_grads else None
        G = np.zeros_like(z) if want_grads else None
        for i, t in enumerate(tt):
            if mode == MIXED:
                tmode = FKL_TOPK if msk[t] == 1 else RKL_MC
            else:
                tmode = mode
            C = k_f if tmode == FKL_TOPK else K_m
            a = idx[t, :C]
            ell = logp[i, a]                               # O3
            old = None if old_all is None else old_all[t, :C]
            L, alpha, beta = token_terms(tmode, lam_all[t, :C], old, ell, flags, surrogate, clip_eps)
            per_token[t] = L
            lse_out[t] = lse[i]
            alpha_out[t] = alpha
            slp[t, :C] = ell
            if tmode == RKL_MC:
                rho_out[t, :C], var1_out[t] = mc_diagnostics(lam_all[t, :C], old, ell)
                first_out[t] = -rho_out[t, 0] * (lam_all[t, 0] - ell[0])
            if want_grads:
                g = alpha * p[i]                           # O7 dense part
                np.add.at(g, a, beta)                      # O7 sparse part (duplicates add)
                G[i] = g * scale
        if want_grads:
            gh[tt] = G @ Wd.T                              # O8
            if gW is not None:
                gW += X[tt].T @ G                          # O9
    loss = float(np.sum(per_token)) * scale                # O6
    return dict(loss=loss, N=N, per_token_kl=per_token, lse=lse_out, student_logp=slp,
                alpha=alpha_out, grad_hidden=gh, grad_W=gW, rho=rho_out, var1=var1_out, first_draw=first_out)


def grad_W_columns(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K,
                   cols, flags: int = 0, norm_override: float = 0.0, chunk: int = 512,
                   surrogate: int = SUR_THETA_NOCLIP, clip_eps: float = 0.2):
    """O9 restricted to the vocabulary columns ``cols``: grad_W[:, cols]  ([d, len(cols)]).

    Every live token contributes to every column, so this still runs O1-O2 for all live tokens.
    ``surrogate`` / ``clip_eps``: the reverse-KL surrogate of Eq.(4),(6),(7), handed to
    ``token_terms`` exactly as ``opd_oracle`` does (pinned against it for all four surrogates).
    """
    X = np.asarray(hidden, dtype=np.float64)
    Wd = np.asarray(W, dtype=np.float64)
    idx = np.asarray(cache_idx).astype(np.int64)
    lam_all = np.asarray(cache_teacher_logp, dtype=np.float64)
    old_all = None if cache_old_logp is None else np.asarray(cache_old_logp, dtype=np.float64)
    msk = np.asarray(mask).astype(np.int64)
    cols = np.asarray(cols, dtype=np.int64)
    T, d = X.shape
    k_f, K_m = _split_k(mode, k_or_K)
    N = float(np.count_nonzero(msk))
    norm = float(norm_override) if norm_override > 0 else N
    scale = 0.0 if norm == 0 else 1.0 / norm
    out = np.zeros((d, cols.size))
    live = np.flatnonzero(msk)
    for s in range(0, live.size, chunk):
        tt = live[s:s + chunk]
        z = X[tt] @ Wd
        logp, _ = log_softmax_rows(z)
        Gc = np.zeros((tt.size, cols.size))
        for i, t in enumerate(tt):
            tmode = (FKL_TOPK if msk[t] == 1 else RKL_MC) if mode == MIXED else mode
            C = k_f if tmode == FKL_TOPK else K_m
            a = idx[t, :C]
            old = None if old_all is None else old_all[t, :C]
            _, alpha, beta = token_terms(tmode, lam_all[t, :C], old, logp[i, a], flags, surrogate, clip_eps)
            g = alpha * np.exp(logp[i, cols])
            for j in range(C):
                g += beta[j] * (cols == a[j])
            Gc[i] = g * scale
        out += X[tt].T @ Gc
    return out


def opd_oracle_loops(hidden, W, cache_idx, cache_teacher_logp, cache_old_logp, mask, mode, k_or_K,
                     flags: int = 0, norm_override: float = 0.0):
    """Same mathematics as ``opd_oracle`` written as plain Python loops over t, k, v (tiny shapes only)."""
    X = [[float(x) for x in row] for row in np.asarray(hidden, dtype=np.float64)]
    Wd = [[float(x) for x in row] for row in np.asarray(W, dtype=np.float64)]
    T, d, V = len(X), len(Wd), len(Wd[0])
    k_f, K_m = _split_k(mode, k_or_K)
    msk = [int(m) for m in np.asarray(mask)]
    N = sum(1 for m in msk if m != 0)
    norm = float(norm_override) if norm_override > 0 else float(N)
    scale = 0.0 if norm == 0 else 1.0 / norm
    per_token = [0.0] * T
    gh = [[0.0] * d for _ in range(T)]
    gW = [[0.0] * V for _ in range(d)]
    for t in range(T):
        if msk[t] == 0:
            continue
        z = [sum(X[t][k] * Wd[k][v] for k in range(d)) for v in range(V)]
        M = max(z)
        lse = M + math.log(sum(math.exp(zv - M) for zv in z))
        logp = [zv - lse for zv in z]
        tmode = (FKL_TOPK if msk[t] == 1 else RKL_MC) if mode == MIXED else mode
        C = k_f if tmode == FKL_TOPK else K_m
        a = [int(cache_idx[t][j]) for j in range(C)]
        lam = [float(cache_teacher_logp[t][j]) for j in range(C)]
        ell = [logp[a[j]] for j in range(C)]
        g = [0.0] * V
        if tmode == FKL_TOPK:
            if flags & F_NO_RENORM_TEACHER:
                logZq = 0.0
            else:
                ml = max(lam)
                logZq = ml + math.log(sum(math.exp(x - ml) for x in lam))
            qt = [math.exp(x - logZq) for x in lam]
            if flags & F_RENORM_STUDENT:
                me = max(ell)
                logZp = me + math.log(sum(math.exp(x - me) for x in ell))
                L = sum(qt[j] * ((lam[j] - logZq) - (ell[j] - logZp)) for j in range(C))
                sq = sum(qt)
                for j in range(C):
                    g[a[j]] += sq * math.exp(ell[j] - logZp) - qt[j]
            else:
                L = sum(qt[j] * ((lam[j] - logZq) - ell[j]) for j in range(C))
                sq = sum(qt)
                for v in range(V):
                    g[v] += sq * math.exp(logp[v])
                for j in range(C):
                    g[a[j]] -= qt[j]
        else:
            old = [float(cache_old_logp[t][j]) for j in range(C)]
            ra = [math.exp(ell[j] - old[j]) * (lam[j] - ell[j]) for j in range(C)]
            c = sum(ra) / C
            L = -c
            for v in range(V):
                g[v] += c * math.exp(logp[v])
            for j in range(C):
                g[a[j]] -= ra[j] / C
        per_token[t] = L
        for k in range(d):
            gh[t][k] = scale * sum(g[v] * Wd[k][v] for v in range(V))
            for v in range(V):
                gW[k][v] += scale * X[t][k] * g[v]
    loss = scale * sum(per_token)
    return dict(loss=loss, N=float(N), per_token_kl=np.array(per_token), grad_hidden=np.array(gh),
                grad_W=np.array(gW))


def mc_diagnostics(lam, old, ell):
    """Per-token diagnostics of the MC estimator: the importance ratios rho_j = p_theta(a_j)/p_old(a_j) whose tail
    Fig. 5 reports, and the unbiased sample variance over the m cached draws of the one-sample
    estimates X_j = -rho_j A_theta,j, i.e. the within-prefix Var(L^MC_1 | s_t) of Eq.(16);
    Var(L^MC_m | s_t) = Var(L^MC_1 | s_t) / m for iid draws. 0 when m = 1."""
    lam = np.asarray(lam, dtype=np.float64); old = np.asarray(old, dtype=np.float64); ell = np.asarray(ell, dtype=np.float64)
    rho = np.exp(ell - old)
    X = -rho * (lam - ell)
    m = X.shape[0]
    var1 = float(np.sum((X - X.mean()) ** 2) / (m - 1)) if m > 1 else 0.0
    return rho, var1


def seq_diagnostics(per_token_mc, first_draw, var1, mask, cu_seqlens, m: int, mc_code=None):
    """Sequence-level diagnostics of App. E, Eq.(17) (Table 6 second column PAPER.md:412-419): "the same
    estimator averaged over generated timesteps".  For every sequence n = token rows [cu[n], cu[n+1]) with T_n live MC rows:

        mean_m[n] = (1/T_n) sum_t L^MC_m(theta; s_t)          (per_token_mc[t], Eq.(15))
        mean_1[n] = (1/T_n) sum_t L^MC_1(theta; s_t)          (first_draw[t] = -rho_t1 A_theta,t1, the first cached draw)
        var_m[n]  = (1/T_n^2) sum_t var1[t] / m               variance of mean_m over the local draws with the prefix path
                                                              fixed: draws are iid across and within prefixes,
                                                              so Var(mean_m) = (1/T_n^2) sum_t Var(L^MC_1 | s_t) / m, with the
                                                              within-prefix variances estimated as in Eq.(16) (mc_diagnostics)
    mc_code: if given (MIXED batches), only rows with mask == mc_code take part; else every live row.
    R_m^seq of Eq.(17) is the ratio of the variances of mean_m and mean_1, which a caller forms over its sequences / batches
    (reading Q19 in DESIGN.md: with the path fixed and iid draws the ratio of the var_m's is exactly 1/m; the paper's measured
    0.338 / 0.152 / 0.112 are above 1/m, i.e. its variance also contains variation that more draws do not remove)."""
    L = np.asarray(per_token_mc, dtype=np.float64)
    L1 = np.asarray(first_draw, dtype=np.float64)
    v1 = np.asarray(var1, dtype=np.float64)
    msk = np.asarray(mask).astype(np.int64)
    cu = np.asarray(cu_seqlens).astype(np.int64)
    n_seq = cu.shape[0] - 1
    mean_m, mean_1, var_m = np.zeros(n_seq), np.zeros(n_seq), np.zeros(n_seq)
    for n in range(n_seq):
        rows = [t for t in range(cu[n], cu[n + 1]) if msk[t] != 0 and (mc_code is None or msk[t] == mc_code)]
        Tn = len(rows)
        if Tn == 0:
            continue
        mean_m[n] = sum(L[t] for t in rows) / Tn
        mean_1[n] = sum(L1[t] for t in rows) / Tn
        var_m[n] = sum(v1[t] for t in rows) / (Tn * Tn * m)
    return mean_m, mean_1, var_m


def sparse_reverse_kl(lam: np.ndarray, ell: np.ndarray):
    """App. A.1 Eq.(8)-(10) for ONE token on a fixed cached support S.

    p~ = softmax(l_j over S), q~ = softmax(lam_j over S); D_R^S = sum_j p~_j (log p~_j - log q~_j).
    Returns (D, dD/dl_j): the support is treated as fixed, the full-vocabulary lse
    cancels, so the gradient is purely sparse: dD/dl_j = p~_j (log p~_j - log q~_j - D).
    """
    lam = np.asarray(lam, dtype=np.float64)
    ell = np.asarray(ell, dtype=np.float64)
    lp = ell - logsumexp(ell)
    lq = lam - logsumexp(lam)
    pt = np.exp(lp)
    D = float(np.sum(pt * (lp - lq)))
    return D, pt * (lp - lq - D)


# ------------------------------------------------------------------------------------------------
# Cache producers: what the scoring / rollout side computes before the learner path.
def cache_topk(hidden, W, k: int):
    """Top-k cache of the scoring model (teacher scores are kept on a finite support; Fig. 1: forward KL is
    teacher-supported):  S_t = TopK(softmax(x_t . W), k), in descending order of probability, ties -> lowest index first
    (a stable sort of the negated logits), with the full-vocabulary log-probs on S_t.
    Returns (idx [T,k] int64, logp [T,k], lse [T], logp_all [T,V])."""
    X = np.asarray(hidden, dtype=np.float64)
    Wd = np.asarray(W, dtype=np.float64)
    z = X @ Wd
    logp, lse = log_softmax_rows(z)
    idx = np.argsort(-z, axis=1, kind="stable")[:, :k]
    return idx, np.take_along_axis(logp, idx, 1), lse, logp


def cache_sample(hidden, W, uniforms):
    """Sample cache of the rollout policy (m local next-token samples per prefix; iid WITH
    replacement from p_old(.|s_t), duplicates allowed), drawn by inverse CDF from given uniforms u_tj in [0,1):
        a_tj = min { v : sum_{v' <= v} p_t(v') >= u_tj * sum_v p_t(v) }
    (the textbook categorical draw; vocabulary order).  Returns (idx [T,K] int64, logp [T,K] = log p_t(a_tj), lse [T],
    cdf [T,V])."""
    X = np.asarray(hidden, dtype=np.float64)
    Wd = np.asarray(W, dtype=np.float64)
    u = np.asarray(uniforms, dtype=np.float64)
    logp, lse = log_softmax_rows(X @ Wd)
    cdf = np.cumsum(np.exp(logp), axis=1)
    T, K = u.shape
    idx = np.empty((T, K), dtype=np.int64)
    for t in range(T):
        idx[t] = np.minimum(np.searchsorted(cdf[t], u[t] * cdf[t, -1], side="left"), cdf.shape[1] - 1)
    return idx, np.take_along_axis(logp, idx, 1), lse, cdf


# ------------------------------------------------------------------------------------------------
# Dense two-head forward KL: the teacher's distribution recomputed from transmitted teacher
# hidden states (the direction PAPER.md:240 names as future work), objective Eq.(1), gradient PAPER.md:59.
def dense_kl_oracle(hidden, W, teacher_hidden, W_T, mask, norm_override: float = 0.0, chunk: int = 512, reverse: bool = False):
    """q_t = softmax(h^T_t . W_T), p_t = softmax(x_t . W);  L_t = sum_v q_tv (log q_tv - log p_tv)  (Eq.(1));
    loss = (1/N) sum_t m_t L_t;  dL_t/dz_tv = (sum_v q_tv) p_tv - q_tv  (= p - q);
    grad_hidden / grad_W by the chain rule (O8, O9).
    reverse=True: the student-weighted direction, Eq.(2):  L_t = sum_v p_tv (log p_tv - log q_tv), whose exact
    gradient in the student logits is  dL_t/dz_tv = p_tv (log p_tv - log q_tv - L_t)  (Eq.(3): the "+1" term
    drops out because sum_v p_v d(log p_v) = 0).
    Returns dict(loss, N, per_token_kl[T], grad_hidden[T,d], grad_W[d,V])."""
    X = np.asarray(hidden, dtype=np.float64)
    Wd = np.asarray(W, dtype=np.float64)
    XT = np.asarray(teacher_hidden, dtype=np.float64)
    WT = np.asarray(W_T, dtype=np.float64)
    msk = np.asarray(mask).astype(np.int64)
    T, d = X.shape
    V = Wd.shape[1]
    N = float(np.count_nonzero(msk))
    norm = float(norm_override) if norm_override > 0 else N
    scale = 0.0 if norm == 0 else 1.0 / norm
    per_token = np.zeros(T)
    gh = np.zeros((T, d))
    gW = np.zeros((d, V))
    live = np.flatnonzero(msk)
    for s in range(0, live.size, chunk):
        tt = live[s:s + chunk]
        logp, _ = log_softmax_rows(X[tt] @ Wd)
        logq, _ = log_softmax_rows(XT[tt] @ WT)
        q = np.exp(logq)
        if reverse:
            pr = np.exp(logp)
            Lt = np.sum(pr * (logp - logq), axis=1)
            per_token[tt] = Lt
            G = pr * (logp - logq - Lt[:, None]) * scale
        else:
            per_token[tt] = np.sum(q * (logq - logp), axis=1)
            G = (np.sum(q, axis=1, keepdims=True) * np.exp(logp) - q) * scale
        gh[tt] = G @ Wd.T
        gW += X[tt].T @ G
    return dict(loss=float(np.sum(per_token)) * scale, N=N, per_token_kl=per_token, grad_hidden=gh, grad_W=gW)


def dense_grad_W_columns(hidden, W, teacher_hidden, W_T, mask, cols, norm_override: float = 0.0, chunk: int = 512,
                         reverse: bool = False):
    """grad_W[:, cols] of ``dense_kl_oracle`` ([d, len(cols)]) without holding the [d,V] gradient: the same per-token logit
    gradients (Eq.(1): p - q;  reverse, Eq.(2),(3) PAPER.md:63-68: p (log p - log q - L_t)), restricted to the
    columns ``cols`` before the contraction with hidden (O9).  Both softmaxes still run over the whole vocabulary."""
    X = np.asarray(hidden, dtype=np.float64)
    Wd = np.asarray(W, dtype=np.float64)
    XT = np.asarray(teacher_hidden, dtype=np.float64)
    WT = np.asarray(W_T, dtype=np.float64)
    msk = np.asarray(mask).astype(np.int64)
    cols = np.asarray(cols, dtype=np.int64)
    N = float(np.count_nonzero(msk))
    norm = float(norm_override) if norm_override > 0 else N
    scale = 0.0 if norm == 0 else 1.0 / norm
    out = np.zeros((X.shape[1], cols.size))
    live = np.flatnonzero(msk)
    for s in range(0, live.size, chunk):
        tt = live[s:s + chunk]
        logp, _ = log_softmax_rows(X[tt] @ Wd)
        logq, _ = log_softmax_rows(XT[tt] @ WT)
        if reverse:
            Lt = np.sum(np.exp(logp) * (logp - logq), axis=1)
            Gc = np.exp(logp[:, cols]) * (logp[:, cols] - logq[:, cols] - Lt[:, None])
        else:
            Gc = np.sum(np.exp(logq), axis=1, keepdims=True) * np.exp(logp[:, cols]) - np.exp(logq[:, cols])
        out += X[tt].T @ (Gc * scale)
    return out

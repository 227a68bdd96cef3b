"""Pins for the fp64 oracle (oracle/opd_oracle.py): what the paper and the mathematics fix.

Each pin names the part of the oracle it fixes (P-numbers as in DESIGN.md "Oracle pins").
None of these tests touches the CUDA path.
"""
import math

import numpy as np
import pytest
import torch

from oracle import opd_oracle as O
from gen import synth


def tiny(seed, T=4, d=6, V=12, C=3, dup=False, mask=None):
    rng = np.random.default_rng(seed)
    X = rng.normal(size=(T, d))
    W = rng.normal(size=(d, V)) / math.sqrt(d)
    WT = rng.normal(size=(d, V)) / math.sqrt(d)
    Wold = W + 0.3 * rng.normal(size=(d, V)) / math.sqrt(d)
    logq, _ = O.log_softmax_rows(X @ WT)
    logpo, _ = O.log_softmax_rows(X @ Wold)
    idx = np.stack([rng.choice(V, size=C, replace=dup) for _ in range(T)])
    if dup:
        idx[:, -1] = idx[:, 0]           # force a duplicate in every row
    lam = np.take_along_axis(logq, idx, 1)
    old = np.take_along_axis(logpo, idx, 1)
    m = np.ones(T, dtype=np.uint8) if mask is None else np.asarray(mask, dtype=np.uint8)
    return dict(X=X, W=W, WT=WT, Wold=Wold, logq=logq, logpo=logpo, idx=idx, lam=lam, old=old, mask=m)


def c1_inputs():
    cfg = dict(synth.CONFIGS[1])
    inp = synth.make_inputs(cfg, c=1, device="cpu", keep_teacher_rows=True)
    f = lambda t: t.to(torch.float64).numpy() if t.is_floating_point() else t.numpy()
    return {k: (f(v) if isinstance(v, torch.Tensor) else v) for k, v in inp.items()}


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("flags", [0, O.F_NO_RENORM_TEACHER, O.F_RENORM_STUDENT,
                                   O.F_NO_RENORM_TEACHER | O.F_RENORM_STUDENT])
def test_P1_topk_with_k_equal_V_is_dense_forward_kl(flags):
    """PAPER.md:57 Eq.(1): the sparse top-k forward KL with S = V is the dense D_F (north_star)."""
    t = tiny(1, T=5, d=7, V=16)
    V = 16
    idx = np.tile(np.arange(V), (5, 1))
    r = O.opd_oracle(t["X"], t["W"], idx, t["logq"], None, t["mask"], O.FKL_TOPK, V, flags=flags)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    DF = O.dense_forward_kl(t["logq"], logp)
    np.testing.assert_allclose(r["per_token_kl"], DF, rtol=0, atol=1e-12)
    assert abs(r["loss"] - DF.mean()) < 1e-12


def test_P1_on_C1_permuted_support():
    c = c1_inputs()
    T, V = 16, c["W"].shape[1]
    rng = np.random.default_rng(0)
    idx = np.stack([rng.permutation(V) for _ in range(T)])
    c["logq"] = O.log_softmax_rows(c["logq"])[0]        # the generator's fp32 rows, renormalised exactly in fp64
    lam = np.take_along_axis(c["logq"][:T], idx, 1)
    r = O.opd_oracle(c["hidden"][:T], c["W"], idx, lam, None, np.ones(T), O.FKL_TOPK, V, want_grads=False)
    logp, _ = O.log_softmax_rows(c["hidden"][:T] @ c["W"])
    np.testing.assert_allclose(r["per_token_kl"], O.dense_forward_kl(c["logq"][:T], logp), atol=1e-11)


# ---------------------------------------------------------------- P2
def test_P2_k1_is_library_cross_entropy_with_softmax_minus_onehot_gradient():
    """k=1 with teacher renorm: L = -log p(a).  Checked end to end against torch's fp64 cross_entropy + autograd."""
    t = tiny(2, T=6, d=5, V=11, C=1)
    r = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], None, t["mask"], O.FKL_TOPK, 1)
    X = torch.tensor(t["X"], requires_grad=True)
    W = torch.tensor(t["W"], requires_grad=True)
    loss = torch.nn.functional.cross_entropy(X @ W, torch.tensor(t["idx"][:, 0]), reduction="mean")
    loss.backward()
    assert abs(r["loss"] - loss.item()) < 1e-12
    np.testing.assert_allclose(r["grad_hidden"], X.grad.numpy(), atol=1e-13)
    np.testing.assert_allclose(r["grad_W"], W.grad.numpy(), atol=1e-13)


# ---------------------------------------------------------------- P3
def test_P3_mc_with_uniform_proposal_over_all_V_is_dense_reverse_kl():
    """Eq.(2),(3),(5) PAPER.md:63-68,128: K=V, a = 0..V-1, o = -log V  =>  L = D_R and the surrogate
    gradient (A frozen) equals the finite-difference gradient of the dense D_R."""
    t = tiny(3, T=3, d=5, V=9)
    V = 9
    idx = np.tile(np.arange(V), (3, 1))
    old = np.full((3, V), -math.log(V))
    r = O.opd_oracle(t["X"], t["W"], idx, t["logq"], old, t["mask"], O.RKL_MC, V)
    def DR(X, W):
        logp, _ = O.log_softmax_rows(X @ W)
        return O.dense_reverse_kl(t["logq"], logp)
    np.testing.assert_allclose(r["per_token_kl"], DR(t["X"], t["W"]), atol=1e-12)
    h = 1e-6
    for (ti, ki) in [(0, 0), (1, 3), (2, 4)]:
        Xp, Xm = t["X"].copy(), t["X"].copy()
        Xp[ti, ki] += h; Xm[ti, ki] -= h
        fd = (DR(Xp, t["W"]).mean() - DR(Xm, t["W"]).mean()) / (2 * h)
        assert abs(fd - r["grad_hidden"][ti, ki]) < 1e-8
    for (ki, vi) in [(0, 0), (2, 5), (4, 8)]:
        Wp, Wm = t["W"].copy(), t["W"].copy()
        Wp[ki, vi] += h; Wm[ki, vi] -= h
        fd = (DR(t["X"], Wp).mean() - DR(t["X"], Wm).mean()) / (2 * h)
        assert abs(fd - r["grad_W"][ki, vi]) < 1e-8


# ---------------------------------------------------------------- P4
def test_P4_importance_sampling_identity_by_enumeration():
    """Eq.(5): sum_a p_old(a) rho(a) A(a) = -D_R for any full-support p_old."""
    t = tiny(4, T=4, d=6, V=10)
    V = 10
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    for ti in range(4):
        tot = 0.0
        for a in range(V):
            L, _, _ = O.token_terms(O.RKL_MC, [t["logq"][ti, a]], [t["logpo"][ti, a]], [logp[ti, a]], 0)
            tot += math.exp(t["logpo"][ti, a]) * L         # L = -rho A for K=1
        DR = O.dense_reverse_kl(t["logq"][ti], logp[ti])
        assert abs(tot - DR) < 1e-12


# ---------------------------------------------------------------- P5 / P12
def test_P5_P12_on_policy_unbiasedness_and_one_over_m_variance():
    """PAPER.md:161, Eq.(11)-(13) PAPER.md:309-317: with p_old = p_theta the estimator's mean converges to D_R;
    PAPER.md:191 + Table 6: Var[L_m] = Var[L_1]/m for iid samples (paper measured
    0.255 / 0.0588 / 0.0149 at m = 4, 16, 64)."""
    t = tiny(5, T=3, d=6, V=14)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    rng = np.random.default_rng(123)
    R = 40000
    for ti in range(3):
        p = np.exp(logp[ti])
        DR = O.dense_reverse_kl(t["logq"][ti], logp[ti])
        var = {}
        for m in (1, 4, 16):
            a = rng.choice(14, size=(R, m), p=p)
            est = np.array([O.token_terms(O.RKL_MC, t["logq"][ti, a[r]], logp[ti, a[r]], logp[ti, a[r]], 0)[0]
                            for r in range(0, R, 8 if m > 1 else 1)])
            se = est.std() / math.sqrt(est.size)
            assert abs(est.mean() - DR) < 5 * se + 1e-12, (m, est.mean(), DR, se)
            var[m] = est.var()
        assert abs(var[4] / var[1] - 0.25) < 0.03
        assert abs(var[16] / var[1] - 1 / 16) < 0.012


def test_P5_stale_proposal_is_still_unbiased_with_IS():
    """Eq.(5): sampling from the generator's stale p_old and weighting by rho is unbiased for D_R."""
    t = tiny(6, T=2, d=6, V=12)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    rng = np.random.default_rng(7)
    for ti in range(2):
        po = np.exp(t["logpo"][ti])
        a = rng.choice(12, size=(30000, 4), p=po / po.sum())
        est = np.array([O.token_terms(O.RKL_MC, t["logq"][ti, r], t["logpo"][ti, r], logp[ti, r], 0)[0] for r in a])
        DR = O.dense_reverse_kl(t["logq"][ti], logp[ti])
        assert abs(est.mean() - DR) < 5 * est.std() / math.sqrt(est.size)


# ---------------------------------------------------------------- P6 / P7
def test_P6_P7_renorm_variants_and_nonnegativity():
    """KL(q~||p) - KL(q~||p~^S) = -log Z_p^S = lse_full - lse_S >= 0; both KLs >= 0 (Gibbs)."""
    c = c1_inputs()
    T = 64
    args = (c["hidden"][:T], c["W"], c["topk_idx"][:T], c["topk_logq"][:T], None, np.ones(T), O.FKL_TOPK, 8)
    a = O.opd_oracle(*args, flags=0, want_grads=False)
    b = O.opd_oracle(*args, flags=O.F_RENORM_STUDENT, want_grads=False)
    lseS = np.array([O.logsumexp(a["student_logp"][t]) for t in range(T)])      # log Z_p^S
    np.testing.assert_allclose(a["per_token_kl"] - b["per_token_kl"], -lseS, atol=1e-12)
    assert (-lseS >= 0).all()
    assert (a["per_token_kl"] >= -1e-15).all() and (b["per_token_kl"] >= -1e-15).all()
    logp, _ = O.log_softmax_rows(c["hidden"][:T] @ c["W"])
    assert (O.dense_forward_kl(c["logq"][:T], logp) >= 0).all()
    assert (O.dense_reverse_kl(c["logq"][:T], logp) >= 0).all()


# ---------------------------------------------------------------- P8
def test_P8_zero_cases_teacher_equals_student():
    t = tiny(8, T=4, d=6, V=12, C=4)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    lam = np.take_along_axis(logp, t["idx"], 1)
    r = O.opd_oracle(t["X"], t["W"], t["idx"], lam, t["old"], t["mask"], O.RKL_MC, 4)
    assert np.all(r["per_token_kl"] == 0) and np.all(r["grad_hidden"] == 0) and np.all(r["grad_W"] == 0)
    f = O.opd_oracle(t["X"], t["W"], t["idx"], lam, None, t["mask"], O.FKL_TOPK, 4)
    lseS = np.array([O.logsumexp(lam[i]) for i in range(4)])
    np.testing.assert_allclose(f["per_token_kl"], -lseS, atol=1e-13)
    full = np.tile(np.arange(12), (4, 1))
    z = O.opd_oracle(t["X"], t["W"], full, logp, None, t["mask"], O.FKL_TOPK, 12)
    assert np.abs(z["per_token_kl"]).max() < 1e-14 and np.abs(z["grad_W"]).max() < 1e-15


# ---------------------------------------------------------------- P9
def _surrogate_loss(t, X, W, mode, C, flags, A_frozen, mask, k_or_K):
    """Loss value recomputed from scratch (independent of token_terms) with MC advantages frozen."""
    logp, _ = O.log_softmax_rows(X @ W)
    N = np.count_nonzero(mask)
    tot = 0.0
    for ti in range(X.shape[0]):
        if mask[ti] == 0:
            continue
        tm = mode if mode != O.MIXED else (O.FKL_TOPK if mask[ti] == 1 else O.RKL_MC)
        Ct = C if mode != O.MIXED else ((k_or_K & 0xFFFF) if tm == O.FKL_TOPK else (k_or_K >> 16))
        a = t["idx"][ti, :Ct]
        ell = logp[ti, a]
        lam = t["lam"][ti, :Ct]
        if tm == O.FKL_TOPK:
            lq = lam if flags & O.F_NO_RENORM_TEACHER else lam - np.log(np.exp(lam).sum())
            lp = ell - np.log(np.exp(ell).sum()) if flags & O.F_RENORM_STUDENT else ell
            tot += float((np.exp(lq) * (lq - lp)).sum())
        else:
            tot += -float((np.exp(ell - t["old"][ti, :Ct]) * A_frozen[ti, :Ct]).mean())
    return tot / N


@pytest.mark.parametrize("mode,flags,dup", [
    (O.FKL_TOPK, 0, False), (O.FKL_TOPK, O.F_NO_RENORM_TEACHER, False), (O.FKL_TOPK, O.F_RENORM_STUDENT, False),
    (O.FKL_TOPK, O.F_RENORM_STUDENT | O.F_NO_RENORM_TEACHER, False),
    (O.RKL_MC, 0, False), (O.RKL_MC, 0, True), (O.MIXED, 0, True)])
def test_P9_central_finite_differences(mode, flags, dup):
    """grad_hidden / grad_W against central differences of an independently written loss; MC uses the
    frozen-A surrogate (stop-gradient)."""
    mask = [1, 0, 2, 1] if mode == O.MIXED else [1, 0, 1, 1]
    t = tiny(9, T=4, d=6, V=12, C=3, dup=dup and mode != O.FKL_TOPK, mask=mask)
    kk = (2 | (3 << 16)) if mode == O.MIXED else 3
    r = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], mode, kk, flags=flags)
    A0 = t["lam"] - np.nan_to_num(r["student_logp"])
    f = lambda X, W: _surrogate_loss(t, X, W, mode, 3, flags, A0, t["mask"], kk)
    h = 1e-6
    rng = np.random.default_rng(0)
    for _ in range(12):
        ti, ki, vi = rng.integers(4), rng.integers(6), rng.integers(12)
        Xp, Xm = t["X"].copy(), t["X"].copy(); Xp[ti, ki] += h; Xm[ti, ki] -= h
        assert abs((f(Xp, t["W"]) - f(Xm, t["W"])) / (2 * h) - r["grad_hidden"][ti, ki]) < 2e-8
        Wp, Wm = t["W"].copy(), t["W"].copy(); Wp[ki, vi] += h; Wm[ki, vi] -= h
        assert abs((f(t["X"], Wp) - f(t["X"], Wm)) / (2 * h) - r["grad_W"][ki, vi]) < 2e-8
    # every cached column is probed too
    for ti in (0, 2, 3):
        vi = int(t["idx"][ti, 0])
        Wp, Wm = t["W"].copy(), t["W"].copy(); Wp[1, vi] += h; Wm[1, vi] -= h
        assert abs((f(t["X"], Wp) - f(t["X"], Wm)) / (2 * h) - r["grad_W"][1, vi]) < 2e-8
    assert np.all(r["grad_hidden"][1] == 0)


# ---------------------------------------------------------------- P10
@pytest.mark.parametrize("mode", [O.FKL_TOPK, O.RKL_MC])
def test_P10_shift_invariance(mode):
    """alpha + sum_j beta_j = 0  =>  every row of g sums to 0  =>  sum_v grad_W[k,v] = 0; adding a constant to a
    row of logits (a ones feature times a constant row of W) leaves the loss unchanged."""
    t = tiny(10, T=5, d=6, V=13, C=4, dup=(mode == O.RKL_MC))
    r = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], mode, 4)
    assert np.abs(r["grad_W"].sum(axis=1)).max() < 1e-14
    X2 = np.concatenate([t["X"], np.ones((5, 1))], axis=1)
    W2 = np.concatenate([t["W"], np.full((1, 13), 3.7)], axis=0)
    r2 = O.opd_oracle(X2, W2, t["idx"], t["lam"], t["old"], t["mask"], mode, 4)
    assert abs(r2["loss"] - r["loss"]) < 1e-12
    np.testing.assert_allclose(r2["grad_W"][:-1], r["grad_W"], atol=1e-13)


# ---------------------------------------------------------------- P11
def test_P11_mask_and_permutations():
    t = tiny(11, T=6, d=5, V=10, C=3, mask=[1, 0, 1, 1, 0, 1])
    base = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], O.RKL_MC, 3)
    X2, lam2, idx2 = t["X"].copy(), t["lam"].copy(), t["idx"].copy()
    X2[[1, 4]] = 1e3; lam2[[1, 4]] = -77.0; idx2[[1, 4]] = 0
    g = O.opd_oracle(X2, t["W"], idx2, lam2, t["old"], t["mask"], O.RKL_MC, 3)
    assert g["loss"] == base["loss"] and np.array_equal(g["grad_W"], base["grad_W"])
    assert np.all(base["grad_hidden"][[1, 4]] == 0) and np.all(base["per_token_kl"][[1, 4]] == 0)
    perm = np.array([3, 0, 5, 1, 2, 4])
    p = O.opd_oracle(t["X"][perm], t["W"], t["idx"][perm], t["lam"][perm], t["old"][perm], t["mask"][perm], O.RKL_MC, 3)
    np.testing.assert_allclose(p["per_token_kl"], base["per_token_kl"][perm], atol=1e-15)
    np.testing.assert_allclose(p["grad_hidden"], base["grad_hidden"][perm], atol=1e-15)
    np.testing.assert_allclose(p["grad_W"], base["grad_W"], atol=1e-14)
    sp = np.array([2, 0, 1])
    s = O.opd_oracle(t["X"], t["W"], t["idx"][:, sp], t["lam"][:, sp], t["old"][:, sp], t["mask"], O.RKL_MC, 3)
    np.testing.assert_allclose(s["per_token_kl"], base["per_token_kl"], atol=1e-15)
    # N = number of live tokens; norm_override rescales
    o = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], O.RKL_MC, 3, norm_override=8.0)
    assert abs(o["loss"] - base["loss"] * 4 / 8) < 1e-15
    z = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], np.zeros(6), O.RKL_MC, 3)
    assert z["loss"] == 0 and np.all(z["grad_W"] == 0)


# ---------------------------------------------------------------- P13
def test_P13_duplicates_and_teacher_constant():
    t = tiny(13, T=4, d=6, V=12, C=1)
    one = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], O.RKL_MC, 1)
    rep = lambda a: np.repeat(a, 5, axis=1)
    five = O.opd_oracle(t["X"], t["W"], rep(t["idx"]), rep(t["lam"]), rep(t["old"]), t["mask"], O.RKL_MC, 5)
    np.testing.assert_allclose(five["per_token_kl"], one["per_token_kl"], atol=1e-14)
    np.testing.assert_allclose(five["grad_W"], one["grad_W"], atol=1e-14)
    u = tiny(14, T=4, d=6, V=12, C=4)
    a = O.opd_oracle(u["X"], u["W"], u["idx"], u["lam"], None, u["mask"], O.FKL_TOPK, 4)
    b = O.opd_oracle(u["X"], u["W"], u["idx"], u["lam"] + np.array([[1.5], [-2.0], [0.3], [9.0]]), None,
                     u["mask"], O.FKL_TOPK, 4)
    np.testing.assert_allclose(a["per_token_kl"], b["per_token_kl"], atol=1e-13)
    np.testing.assert_allclose(a["grad_hidden"], b["grad_hidden"], atol=1e-14)


# ---------------------------------------------------------------- P14
@pytest.mark.parametrize("mode,flags", [(O.FKL_TOPK, 0), (O.FKL_TOPK, O.F_RENORM_STUDENT), (O.RKL_MC, 0), (O.MIXED, 0)])
def test_P14_loops_agree_with_vectorised(mode, flags):
    mask = [2, 1, 0, 1, 2] if mode == O.MIXED else [1, 1, 0, 1, 1]
    t = tiny(15, T=5, d=4, V=9, C=3, dup=(mode != O.FKL_TOPK), mask=mask)
    kk = (3 | (2 << 16)) if mode == O.MIXED else 3
    a = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], mode, kk, flags=flags, chunk=2)
    b = O.opd_oracle_loops(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], mode, kk, flags=flags)
    assert abs(a["loss"] - b["loss"]) < 1e-13
    np.testing.assert_allclose(a["grad_hidden"], b["grad_hidden"], atol=1e-13)
    np.testing.assert_allclose(a["grad_W"], b["grad_W"], atol=1e-13)
    cols = [0, 4, int(t["idx"][0, 0]), 8]
    gc = O.grad_W_columns(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], mode, kk, cols, flags=flags)
    np.testing.assert_allclose(gc, b["grad_W"][:, cols], atol=1e-13)
    sub = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], mode, kk, flags=flags, rows=[0, 3])
    np.testing.assert_allclose(sub["grad_hidden"][[0, 3]], b["grad_hidden"][[0, 3]], atol=1e-13)


# ---------------------------------------------------------------- NEXT-1 / NEXT-2 pins
def test_surrogate_variants_reduce_to_reference():
    """Eq.(6),(7) PAPER.md:132-141: with eps -> inf the clipped forms equal the unclipped ones; with W_old = W
    (rho = 1, A_old = A_theta) all four coincide."""
    t = tiny(16, T=3, d=5, V=10, C=4)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    for ti in range(3):
        ell = logp[ti, t["idx"][ti]]
        ref = O.token_terms(O.RKL_MC, t["lam"][ti], t["old"][ti], ell, 0, O.SUR_THETA_NOCLIP)
        big = O.token_terms(O.RKL_MC, t["lam"][ti], t["old"][ti], ell, 0, O.SUR_THETA_CLIP, clip_eps=1e9)
        assert abs(ref[0] - big[0]) < 1e-15 and np.allclose(ref[2], big[2], atol=1e-15)
        same = [O.token_terms(O.RKL_MC, t["lam"][ti], ell, ell, 0, s) for s in range(4)]
        for s in same[1:]:
            assert abs(s[0] - same[0][0]) < 1e-15 and np.allclose(s[2], same[0][2], atol=1e-15)
        # clipped objective never exceeds... min(.,.) <= unclipped term, so L_clip >= L_noclip
        cl = O.token_terms(O.RKL_MC, t["lam"][ti], t["old"][ti], ell, 0, O.SUR_OLD_CLIP, clip_eps=0.2)
        nc = O.token_terms(O.RKL_MC, t["lam"][ti], t["old"][ti], ell, 0, O.SUR_OLD_NOCLIP)
        assert cl[0] >= nc[0] - 1e-15


def _clip_case(seed=71, T=4, d=6, V=12, C=6):
    """Inputs on which old != ell, A_old != A_theta, and the PPO clip bites in BOTH directions: every row holds slots with
    rho > 1+eps and rho < 1-eps, each with advantages of both signs (checked by the caller)."""
    t = tiny(seed, T=T, d=d, V=V, C=C, dup=True, mask=[1, 0, 1, 1])
    rng = np.random.default_rng(seed)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    ell = np.take_along_axis(logp, t["idx"], 1)
    # rollout-time log-probs placed so that rho = exp(ell - old) lands on both sides of the clip range, away from its edges
    shift = np.array([0.9, -0.9, 0.45, -0.45, 0.05, -0.07])[:C]
    t["old"] = ell - np.stack([rng.permutation(shift) for _ in range(T)])
    # teacher scores around both log-probs so that A_theta and A_old take both signs and differ
    t["lam"] = 0.5 * (ell + t["old"]) + rng.normal(size=ell.shape) * 0.8
    return t, ell


def _ppo_surrogate_from_scratch(X, W, t, A_frozen, clip, eps=0.2):
    """Eq.(4) / Eq.(6),(7) written out with the expectation over a ~ p_old replaced by the mean over
    the m cached draws (Eq.(15)):  L = (1/N) sum_t -(1/m) sum_j min(rho_j A_j, clip(rho_j, 1-eps, 1+eps) A_j),
    rho_j = p_theta(a_j) / p_old(a_j); without clipping the clipped term is dropped.  A is a constant here
    (stop-gradient): the caller passes A_old = log q - log p_old or A_theta frozen at the base point."""
    tot, N = 0.0, 0
    for ti in range(X.shape[0]):
        if t["mask"][ti] == 0:
            continue
        N += 1
        z = X[ti] @ W
        lse = math.log(sum(math.exp(v) for v in z))
        acc = 0.0
        m = t["idx"].shape[1]
        for j in range(m):
            rho = math.exp(z[t["idx"][ti, j]] - lse - t["old"][ti, j])
            a = A_frozen[ti, j]
            if clip:
                acc += min(rho * a, min(max(rho, 1.0 - eps), 1.0 + eps) * a)
            else:
                acc += rho * a
        tot += -acc / m
    return tot / N


@pytest.mark.parametrize("sur", [O.SUR_THETA_NOCLIP, O.SUR_THETA_CLIP, O.SUR_OLD_NOCLIP, O.SUR_OLD_CLIP])
def test_surrogates_against_eq4_eq6_eq7_written_out(sur):
    """NEXT-1 pins: value of each of the four surrogates against Eq.(6)/(7) written from scratch (1e-13) and its gradients
    against central differences of that frozen-A surrogate, on inputs where p_old != p_theta and the clip is active in both
    directions.  An oracle that ignored the A_old flag, or that let gradient through clipped slots, fails here."""
    t, ell = _clip_case()
    live = t["mask"] != 0
    rho = np.exp(ell - t["old"])
    A_th, A_old = t["lam"] - ell, t["lam"] - t["old"]
    for A in (A_th, A_old):                          # the case really exercises all four corners of the clip
        assert ((rho > 1.2) & (A > 0))[live].any() and ((rho > 1.2) & (A < 0))[live].any()
        assert ((rho < 0.8) & (A > 0))[live].any() and ((rho < 0.8) & (A < 0))[live].any()
    assert np.abs(np.abs(rho - 1.0) - 0.2).min() > 1e-3       # no slot sits on a clip edge (finite differences are valid)
    use_old = sur in (O.SUR_OLD_NOCLIP, O.SUR_OLD_CLIP)
    clip = sur in (O.SUR_THETA_CLIP, O.SUR_OLD_CLIP)
    A0 = A_old if use_old else A_th
    r = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], O.RKL_MC, t["idx"].shape[1], surrogate=sur)
    f = lambda X, W: _ppo_surrogate_from_scratch(X, W, t, A0, clip)
    assert abs(r["loss"] - f(t["X"], t["W"])) < 1e-13
    # discriminating power of the value pin: the other advantage / the other clipping give a different number
    assert abs(f(t["X"], t["W"]) - _ppo_surrogate_from_scratch(t["X"], t["W"], t, A_th if use_old else A_old, clip)) > 1e-2
    assert abs(f(t["X"], t["W"]) - _ppo_surrogate_from_scratch(t["X"], t["W"], t, A0, not clip)) > 1e-2
    h = 1e-6
    rng = np.random.default_rng(5)
    probes = [(int(rng.integers(4)), int(rng.integers(6)), int(rng.integers(12))) for _ in range(10)]
    probes += [(ti, 3, int(t["idx"][ti, j])) for ti in (0, 2, 3) for j in range(t["idx"].shape[1])]
    worst_noclip_gap = 0.0
    rn = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], O.RKL_MC, t["idx"].shape[1],
                      surrogate=O.SUR_OLD_NOCLIP if use_old else O.SUR_THETA_NOCLIP)
    for ti, ki, vi in probes:
        Xp, Xm = t["X"].copy(), t["X"].copy(); Xp[ti, ki] += h; Xm[ti, ki] -= h
        fd = (f(Xp, t["W"]) - f(Xm, t["W"])) / (2 * h)
        assert abs(fd - r["grad_hidden"][ti, ki]) < 2e-8
        Wp, Wm = t["W"].copy(), t["W"].copy(); Wp[ki, vi] += h; Wm[ki, vi] -= h
        fd = (f(t["X"], Wp) - f(t["X"], Wm)) / (2 * h)
        assert abs(fd - r["grad_W"][ki, vi]) < 2e-8
        worst_noclip_gap = max(worst_noclip_gap, abs(fd - rn["grad_W"][ki, vi]))
    if clip:        # dropping the clip's "active" mask from the gradient would give the unclipped gradient: visibly different
        assert worst_noclip_gap > 1e-3
    assert np.all(r["grad_hidden"][1] == 0)


def test_clipped_surrogate_slot_by_slot():
    """Eq.(4) PAPER.md:72 slot by slot through token_terms (K = 1): in the two clipped corners (rho > 1+eps with A > 0,
    rho < 1-eps with A < 0) the term is the constant clip(rho) A and carries no gradient; in the other two the unclipped
    term rho A is the minimum and the gradient is that of rho A (beta = -rho A, alpha = rho A)."""
    for rho, A in [(1.5, 0.7), (0.6, -0.4), (1.5, -0.7), (0.6, 0.4), (1.1, 0.3), (0.9, -0.3)]:
        ell, old = -2.0, -2.0 - math.log(rho)
        for sur, lam in ((O.SUR_THETA_CLIP, ell + A), (O.SUR_OLD_CLIP, old + A)):
            L, alpha, beta = O.token_terms(O.RKL_MC, [lam], [old], [ell], 0, sur)
            clipped = (rho > 1.2 and A > 0) or (rho < 0.8 and A < 0)
            want = -(min(max(rho, 0.8), 1.2) * A) if clipped else -(rho * A)
            assert abs(L - want) < 1e-15
            assert abs(alpha - (0.0 if clipped else rho * A)) < 1e-15 and abs(beta[0] + alpha) < 1e-15


def test_sparse_reverse_kl_definition_and_gradient():
    """Eq.(9),(10) PAPER.md:293-301: S = V gives dense D_R; gradient by finite differences; D >= 0."""
    t = tiny(17, T=2, d=5, V=8)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    D, g = O.sparse_reverse_kl(t["logq"][0], logp[0])
    assert abs(D - O.dense_reverse_kl(t["logq"][0], logp[0])) < 1e-13
    lam, ell = t["logq"][1, :5] + 0.4, logp[1, :5]
    D, g = O.sparse_reverse_kl(lam, ell)
    assert D >= 0
    for j in range(5):
        e = np.zeros(5); e[j] = 1e-6
        fd = (O.sparse_reverse_kl(lam, ell + e)[0] - O.sparse_reverse_kl(lam, ell - e)[0]) / 2e-6
        assert abs(fd - g[j]) < 1e-9


def _rkl_topk_loss(t, X, W, C, mask):
    """Eq.(10) PAPER.md:297-301 from scratch: token mean of KL(p~^S || q~^S) on the fixed cached support."""
    logp, _ = O.log_softmax_rows(X @ W)
    tot = 0.0
    for ti in range(X.shape[0]):
        if mask[ti] == 0:
            continue
        a = t["idx"][ti, :C]
        pt = np.exp(logp[ti, a]); pt = pt / pt.sum()
        qt = np.exp(t["lam"][ti, :C]); qt = qt / qt.sum()
        tot += float((pt * (np.log(pt) - np.log(qt))).sum())
    return tot / np.count_nonzero(mask)


def test_rkl_topk_end_to_end():
    """OPD_RKL_TOPK through opd_oracle: S = V equals dense D_R (Eq.(2)); loss and gradients against central
    differences of an independently written Eq.(10); non-negative; invariant to a per-token teacher constant."""
    t = tiny(23, T=4, d=6, V=12, C=4, mask=[1, 0, 1, 1])
    full = np.tile(np.arange(12), (4, 1))
    r = O.opd_oracle(t["X"], t["W"], full, t["logq"], None, t["mask"], O.RKL_TOPK, 12)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    live = t["mask"] != 0
    assert np.abs(r["per_token_kl"][live] - O.dense_reverse_kl(t["logq"], logp)[live]).max() < 1e-13
    r = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], None, t["mask"], O.RKL_TOPK, 4)
    f = lambda X, W: _rkl_topk_loss(t, X, W, 4, t["mask"])
    assert abs(r["loss"] - f(t["X"], t["W"])) < 1e-14 and np.all(r["per_token_kl"] >= 0)
    h = 1e-6
    rng = np.random.default_rng(1)
    probes = [(int(rng.integers(4)), int(rng.integers(6)), int(rng.integers(12))) for _ in range(10)]
    probes += [(ti, 2, int(t["idx"][ti, j])) for ti in (0, 2, 3) for j in range(4)]
    for ti, ki, vi in probes:
        Xp, Xm = t["X"].copy(), t["X"].copy(); Xp[ti, ki] += h; Xm[ti, ki] -= h
        assert abs((f(Xp, t["W"]) - f(Xm, t["W"])) / (2 * h) - r["grad_hidden"][ti, ki]) < 2e-8
        Wp, Wm = t["W"].copy(), t["W"].copy(); Wp[ki, vi] += h; Wm[ki, vi] -= h
        assert abs((f(t["X"], Wp) - f(t["X"], Wm)) / (2 * h) - r["grad_W"][ki, vi]) < 2e-8
    assert np.all(r["grad_hidden"][1] == 0)
    r2 = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"] + 1.7, None, t["mask"], O.RKL_TOPK, 4)
    assert abs(r2["loss"] - r["loss"]) < 1e-14
    # columns outside the support get no gradient (purely sparse backward)
    outside = np.setdiff1d(np.arange(12), np.unique(t["idx"][live]))
    assert np.all(r["grad_W"][:, outside] == 0)


def test_mc_diagnostics():
    """rho == 1 on-policy (W_old = W); var1 is numpy's unbiased variance of the one-sample estimates
    written out from Eq.(15); the m-sample estimate is their mean, so its within-prefix variance is var1 / m."""
    t = tiny(31, T=3, d=5, V=9, C=4, dup=True)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    on = np.take_along_axis(logp, t["idx"], 1)
    r = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], on, t["mask"], O.RKL_MC, 4)
    assert np.abs(r["rho"] - 1).max() < 1e-14
    r = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], t["old"], t["mask"], O.RKL_MC, 4)
    for ti in range(3):
        ell = logp[ti, t["idx"][ti]]
        x = [-math.exp(ell[j] - t["old"][ti, j]) * (t["lam"][ti, j] - ell[j]) for j in range(4)]
        assert abs(r["var1"][ti] - np.var(x, ddof=1)) < 1e-13
        assert abs(r["per_token_kl"][ti] - np.mean(x)) < 1e-14
        assert np.abs(r["rho"][ti] - np.exp(ell - t["old"][ti])).max() < 1e-14
    r1 = O.opd_oracle(t["X"], t["W"], t["idx"][:, :1], t["lam"][:, :1], t["old"][:, :1], t["mask"], O.RKL_MC, 1)
    assert np.all(r1["var1"] == 0)


def test_seq_diagnostics_by_enumeration():
    """Eq.(17) PAPER.md:388-390 on a 2-token toy sequence: enumerating every pair of m-tuples of local draws (prefix path
    fixed) gives the exact variance of the sequence mean of L^MC_m; the oracle's var_m is an unbiased
    estimate of it (its expectation over all draws equals it), its mean_m / mean_1 average to the mean dense reverse KL
    (Eq.(5)), and the ratio of the fixed-path variances is 1/m."""
    import itertools
    t = tiny(81, T=2, d=4, V=4)
    V, m = 4, 2
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    po = np.exp(t["logpo"])
    DR = O.dense_reverse_kl(t["logq"], logp)
    tuples = list(itertools.product(range(V), repeat=m))
    E_mean_m = E_mean_1 = E_sq = E_sq1 = E_var = 0.0
    for a0 in tuples:
        for a1 in tuples:
            idx = np.array([a0, a1])
            pr = float(np.prod(po[0, list(a0)]) * np.prod(po[1, list(a1)]))
            lam = np.take_along_axis(t["logq"], idx, 1)
            old = np.take_along_axis(t["logpo"], idx, 1)
            r = O.opd_oracle(t["X"], t["W"], idx, lam, old, np.ones(2), O.RKL_MC, m, want_grads=False)
            mm, m1, vm = O.seq_diagnostics(r["per_token_kl"], r["first_draw"], r["var1"], np.ones(2), [0, 2], m)
            # the pieces, written out: L_m per token is the mean of the per-draw terms, L_1 the first of them
            x = [[-math.exp(logp[ti, a] - t["logpo"][ti, a]) * (t["logq"][ti, a] - logp[ti, a]) for a in idx[ti]] for ti in range(2)]
            assert abs(mm[0] - 0.5 * (np.mean(x[0]) + np.mean(x[1]))) < 1e-14 and abs(m1[0] - 0.5 * (x[0][0] + x[1][0])) < 1e-14
            E_mean_m += pr * mm[0]; E_mean_1 += pr * m1[0]; E_sq += pr * mm[0] ** 2; E_sq1 += pr * m1[0] ** 2; E_var += pr * vm[0]
    assert abs(E_mean_m - DR.mean()) < 1e-12 and abs(E_mean_1 - DR.mean()) < 1e-12          # Eq.(5), averaged over the sequence
    var_m, var_1 = E_sq - E_mean_m ** 2, E_sq1 - E_mean_1 ** 2
    assert abs(E_var - var_m) < 1e-12                                                        # unbiased estimate of Var(mean_m)
    assert abs(var_m / var_1 - 1.0 / m) < 1e-10                                              # fixed path, iid draws: exactly 1/m
    # rows outside the sequence, masked rows and (MIXED) non-MC rows do not take part; empty sequences give zeros
    mm, m1, vm = O.seq_diagnostics([1.0, 2.0, 4.0, 8.0], [1.0, 1.0, 1.0, 1.0], [0.5, 0.5, 0.5, 0.5], [2, 1, 0, 2], [0, 3, 3, 4], 4, mc_code=2)
    assert np.allclose(mm, [1.0, 0.0, 8.0]) and np.allclose(vm, [0.5 / 4, 0.0, 0.5 / 4])


def test_cache_topk_against_library_topk_and_ties():
    """cache_topk: values equal torch.topk's (library routine), the set is the k largest, k = V is a full
    descending sort, exact ties resolve to the lowest index."""
    t = tiny(41, T=5, d=6, V=40)
    idx, lp, lse, logp = O.cache_topk(t["X"], t["W"], 7)
    tv, ti = torch.topk(torch.from_numpy(logp), 7, dim=1)
    assert np.allclose(lp, tv.numpy(), atol=1e-15) and np.array_equal(idx, ti.numpy())
    for r in range(5):
        rest = np.delete(logp[r], idx[r])
        assert rest.max() <= lp[r].min() and np.all(np.diff(lp[r]) <= 0)
    assert abs(np.exp(O.cache_topk(t["X"], t["W"], 40)[1]).sum(1) - 1).max() < 1e-12
    W2 = t["W"].copy(); W2[:, 30] = W2[:, 3]; W2[:, 17] = W2[:, 3]          # three exactly tied columns
    idx2 = O.cache_topk(t["X"], W2, 40)[0]
    for r in range(5):
        pos = [int(np.flatnonzero(idx2[r] == c)[0]) for c in (3, 17, 30)]
        assert pos[1] == pos[0] + 1 and pos[2] == pos[0] + 2


def test_cache_sample_is_the_inverse_cdf_draw():
    """cache_sample against a brute-force scan, the frequency law on a uniform grid (counts of
    index v = p_v * n up to 1), u -> 0 / 1 edges, and duplicates being allowed."""
    t = tiny(43, T=3, d=5, V=11)
    rng = np.random.default_rng(2)
    u = rng.random((3, 6))
    idx, lp, lse, cdf = O.cache_sample(t["X"], t["W"], u)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    p = np.exp(logp)
    for r in range(3):
        for j in range(6):
            acc, v = 0.0, 0
            while True:
                acc += p[r, v]
                if acc >= u[r, j] * p[r].sum() or v == 10:
                    break
                v += 1
            assert v == idx[r, j] and abs(lp[r, j] - logp[r, v]) < 1e-15
    n = 20000
    grid = np.tile((np.arange(n) + 0.5) / n, (3, 1))
    gi = O.cache_sample(t["X"], t["W"], grid)[0]
    for r in range(3):
        assert np.abs(np.bincount(gi[r], minlength=11) - p[r] * n).max() <= 1.0 + 1e-9
    e = O.cache_sample(t["X"], t["W"], np.array([[0.0, 1.0 - 1e-16]] * 3))[0]
    assert np.all(e[:, 0] == 0) and np.all(e[:, 1] == 10)
    same = O.cache_sample(t["X"], t["W"], np.full((3, 4), 0.37))[0]
    assert np.all(same == same[:, :1])


def test_P12_paper_table6_fixed_prefix_ratios_follow_one_over_m():
    """tests/golden/paper_table6_mc_variance_ratios.txt (Table 6): the paper's measured fixed-prefix
    ratios R_m^local sit within 7% of 1/m; the oracle's estimator obeys the same law exactly in expectation, which its
    within-prefix diagnostics reproduce: E[var of the m-sample mean] = var1 / m (mc_diagnostics), here checked by
    enumeration of all m-tuples of a small categorical."""
    import itertools
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "paper_table6_mc_variance_ratios.txt"))
            if l.strip() and not l.startswith("#")]
    table = {int(r[0]): float(r[1]) for r in rows}
    for m, ratio in table.items():
        assert abs(ratio * m - 1.0) < 0.07
    t = tiny(51, T=1, d=4, V=5)
    logp, _ = O.log_softmax_rows(t["X"] @ t["W"])
    po = np.exp(t["logpo"][0])
    def var_of_mean(m):
        mean = sq = 0.0
        for a in itertools.product(range(5), repeat=m):
            a = np.array(a)
            pr = float(np.prod(po[a]))
            L = O.token_terms(O.RKL_MC, t["logq"][0, a], t["logpo"][0, a], logp[0, a], 0)[0]
            mean += pr * L; sq += pr * L * L
        return sq - mean * mean
    v1 = var_of_mean(1)
    for m in (2, 4):
        assert abs(var_of_mean(m) / v1 - 1.0 / m) < 1e-10


def test_dense_two_head_kl_pins():
    """dense_kl_oracle (Eq.(1)): equals torch's kl_div (library) and its autograd gradients; equals the
    top-k forward KL at k = V fed with the teacher's full log-probs (pin P1's relation, through opd_oracle); zero when
    the two heads coincide; central finite differences; masked rows contribute nothing."""
    t = tiny(61, T=5, d=6, V=13, mask=[1, 1, 0, 1, 1])
    rng = np.random.default_rng(4)
    XT = rng.normal(size=(5, 8)); WT = rng.normal(size=(8, 13)) / math.sqrt(8)
    r = O.dense_kl_oracle(t["X"], t["W"], XT, WT, t["mask"])
    X = torch.tensor(t["X"], requires_grad=True); W = torch.tensor(t["W"], requires_grad=True)
    logp = torch.log_softmax(X @ W, dim=1)
    logq = torch.log_softmax(torch.tensor(XT) @ torch.tensor(WT), dim=1)
    m = torch.tensor(t["mask"] != 0)
    per = torch.nn.functional.kl_div(logp, logq, reduction="none", log_target=True).sum(1)
    loss = per[m].sum() / m.sum()
    loss.backward()
    assert abs(r["loss"] - loss.item()) < 1e-14 and np.abs(r["per_token_kl"][m.numpy()] - per[m].detach().numpy()).max() < 1e-14
    assert np.abs(r["grad_hidden"] - X.grad.numpy()).max() < 1e-14 and np.abs(r["grad_W"] - W.grad.numpy()).max() < 1e-14
    assert np.all(r["grad_hidden"][2] == 0) and r["per_token_kl"][2] == 0
    full = np.tile(np.arange(13), (5, 1))
    r2 = O.opd_oracle(t["X"], t["W"], full, logq.numpy(), None, t["mask"], O.FKL_TOPK, 13)
    assert abs(r2["loss"] - r["loss"]) < 1e-13 and np.abs(r2["grad_W"] - r["grad_W"]).max() < 1e-14
    z = O.dense_kl_oracle(t["X"], t["W"], t["X"], t["W"], t["mask"])
    assert abs(z["loss"]) < 1e-15 and np.abs(z["grad_W"]).max() < 1e-15
    f = lambda Xa, Wa: O.dense_kl_oracle(Xa, Wa, XT, WT, t["mask"])["loss"]
    h = 1e-6
    for ti, ki, vi in [(0, 1, 2), (3, 5, 12), (4, 0, 7)]:
        Xp, Xm = t["X"].copy(), t["X"].copy(); Xp[ti, ki] += h; Xm[ti, ki] -= h
        assert abs((f(Xp, t["W"]) - f(Xm, t["W"])) / (2 * h) - r["grad_hidden"][ti, ki]) < 2e-8
        Wp, Wm = t["W"].copy(), t["W"].copy(); Wp[ki, vi] += h; Wm[ki, vi] -= h
        assert abs((f(t["X"], Wp) - f(t["X"], Wm)) / (2 * h) - r["grad_W"][ki, vi]) < 2e-8


def test_dense_two_head_reverse_kl_pins():
    """dense_kl_oracle(reverse=True) (Eq.(2); gradient Eq.(3)): equals torch's kl_div with the
    roles swapped (library) and its autograd gradients; equals the MC estimator with K = V and a uniform proposal (pin P3's
    relation) and the sparse reverse KL on S = V, through opd_oracle; zero when the heads coincide; >= 0; central finite
    differences; masked rows contribute nothing."""
    t = tiny(62, T=5, d=6, V=13, mask=[1, 0, 1, 1, 1])
    rng = np.random.default_rng(6)
    XT = rng.normal(size=(5, 8)); WT = rng.normal(size=(8, 13)) / math.sqrt(8)
    r = O.dense_kl_oracle(t["X"], t["W"], XT, WT, t["mask"], reverse=True)
    X = torch.tensor(t["X"], requires_grad=True); W = torch.tensor(t["W"], requires_grad=True)
    logp = torch.log_softmax(X @ W, dim=1)
    logq = torch.log_softmax(torch.tensor(XT) @ torch.tensor(WT), dim=1)
    m = torch.tensor(t["mask"] != 0)
    per = torch.nn.functional.kl_div(logq, logp, reduction="none", log_target=True).sum(1)      # sum_v p (log p - log q)
    loss = per[m].sum() / m.sum()
    loss.backward()
    assert abs(r["loss"] - loss.item()) < 1e-14 and np.abs(r["per_token_kl"][m.numpy()] - per[m].detach().numpy()).max() < 1e-14
    assert np.abs(r["grad_hidden"] - X.grad.numpy()).max() < 1e-14 and np.abs(r["grad_W"] - W.grad.numpy()).max() < 1e-14
    assert np.all(r["grad_hidden"][1] == 0) and r["per_token_kl"][1] == 0 and np.all(r["per_token_kl"] >= 0)
    full = np.tile(np.arange(13), (5, 1))
    lq = logq.numpy()
    mc = O.opd_oracle(t["X"], t["W"], full, lq, np.full((5, 13), -math.log(13)), t["mask"], O.RKL_MC, 13)
    assert abs(mc["loss"] - r["loss"]) < 1e-13 and np.abs(mc["grad_W"] - r["grad_W"]).max() < 1e-13
    sp = O.opd_oracle(t["X"], t["W"], full, lq, None, t["mask"], O.RKL_TOPK, 13)
    assert abs(sp["loss"] - r["loss"]) < 1e-13 and np.abs(sp["grad_hidden"] - r["grad_hidden"]).max() < 1e-13
    z = O.dense_kl_oracle(t["X"], t["W"], t["X"], t["W"], t["mask"], reverse=True)
    assert abs(z["loss"]) < 1e-15 and np.abs(z["grad_W"]).max() < 1e-15
    f = lambda Xa, Wa: O.dense_kl_oracle(Xa, Wa, XT, WT, t["mask"], reverse=True)["loss"]
    h = 1e-6
    for ti, ki, vi in [(0, 1, 2), (3, 5, 12), (4, 0, 7)]:
        Xp, Xm = t["X"].copy(), t["X"].copy(); Xp[ti, ki] += h; Xm[ti, ki] -= h
        assert abs((f(Xp, t["W"]) - f(Xm, t["W"])) / (2 * h) - r["grad_hidden"][ti, ki]) < 2e-8
        Wp, Wm = t["W"].copy(), t["W"].copy(); Wp[ki, vi] += h; Wm[ki, vi] -= h
        assert abs((f(t["X"], Wp) - f(t["X"], Wm)) / (2 * h) - r["grad_W"][ki, vi]) < 2e-8
    # the two directions differ (a swapped-roles mistake would show)
    assert abs(O.dense_kl_oracle(t["X"], t["W"], XT, WT, t["mask"])["loss"] - r["loss"]) > 1e-3


# ---------------------------------------------------------------- column-restricted gradients used by the full-size GPU checks
@pytest.mark.parametrize("mode", [O.RKL_MC, O.MIXED])
def test_grad_W_columns_with_surrogates_equals_the_full_oracle(mode):
    """grad_W_columns(surrogate=s) is opd_oracle(surrogate=s)["grad_W"][:, cols] for the four surrogates of Eq.(6),(7)
    (PAPER.md:132-141), on a stale cache (rho far from 1) where the four gradients really differ from one another."""
    mask = [2, 1, 0, 2, 2, 1, 2, 2] if mode == O.MIXED else [1, 1, 0, 1, 1, 1, 1, 1]
    t = tiny(41, T=8, d=5, V=11, C=4, dup=True, mask=mask)
    old = t["old"] + np.random.default_rng(5).normal(size=t["old"].shape) * 0.6        # heavy importance-ratio tails
    kk = (3 | (4 << 16)) if mode == O.MIXED else 4
    cols = [0, 3, int(t["idx"][0, 0]), int(t["idx"][3, 1]), 10]
    seen = []
    for sur in (O.SUR_THETA_NOCLIP, O.SUR_THETA_CLIP, O.SUR_OLD_NOCLIP, O.SUR_OLD_CLIP):
        full = O.opd_oracle(t["X"], t["W"], t["idx"], t["lam"], old, t["mask"], mode, kk, surrogate=sur, norm_override=3.0)
        gc = O.grad_W_columns(t["X"], t["W"], t["idx"], t["lam"], old, t["mask"], mode, kk, cols, surrogate=sur, norm_override=3.0,
                              chunk=3)
        np.testing.assert_allclose(gc, full["grad_W"][:, cols], atol=1e-13)
        seen.append(gc)
    for i in range(4):
        for j in range(i + 1, 4):
            assert np.abs(seen[i] - seen[j]).max() > 1e-3          # a dropped `surrogate` argument would not pass


@pytest.mark.parametrize("reverse", [False, True])
def test_dense_grad_W_columns_equals_the_full_dense_oracle(reverse):
    """dense_grad_W_columns is dense_kl_oracle(...)["grad_W"][:, cols] in both directions (Eq.(1) / Eq.(2),(3)),
    with masked rows, a normaliser override and a chunk size that does not divide the live count."""
    rng = np.random.default_rng(43)
    T, d, dT, V = 9, 5, 7, 13
    X, XT = rng.normal(size=(T, d)), rng.normal(size=(T, dT))
    W, WT = rng.normal(size=(d, V)) / math.sqrt(d), rng.normal(size=(dT, V)) / math.sqrt(dT)
    mask = np.array([1, 1, 0, 1, 1, 1, 0, 1, 1])
    cols = [0, 5, 12, 7]
    full = O.dense_kl_oracle(X, W, XT, WT, mask, norm_override=4.0, reverse=reverse)
    gc = O.dense_grad_W_columns(X, W, XT, WT, mask, cols, norm_override=4.0, chunk=4, reverse=reverse)
    np.testing.assert_allclose(gc, full["grad_W"][:, cols], atol=1e-13)
    other = O.dense_grad_W_columns(X, W, XT, WT, mask, cols, norm_override=4.0, reverse=not reverse)
    assert np.abs(gc - other).max() > 1e-3                          # the two directions are not interchangeable

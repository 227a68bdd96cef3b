"""GPU parity of the cache producers (opd_cache_topk / opd_cache_sample) against the fp64 oracle.

Floating point decides integers here (which index is the k-th largest, which index a uniform falls on), so the
comparison is: exact agreement wherever the fp64 decision has a margin, and VALIDITY everywhere (the chosen index is a
correct answer within the fp32 resolution of the kernel's logits / cumulative sums)."""
import numpy as np
import pytest
import torch

from oracle import opd_oracle as O
from gen import synth
from tests._util import LOGP_ATOL, f64

pytestmark = pytest.mark.gpu
DEV = "cuda"
ZTOL = 1e-4        # fp32-accumulated logits against fp64 (same bound as LOGP_ATOL)
CDF_TOL = 2e-5     # fp32 cumulative probabilities over up to 1.5e5 terms


@pytest.fixture(scope="module")
def handle():
    from paper_2606_24143_b200 import opd
    return opd.Handle(0)


def inputs(dtype, T, d, V, seed, scale=1.0):
    g = torch.Generator(device=DEV).manual_seed(synth.SEED0 + seed)
    dt = torch.bfloat16 if dtype == "bf16" else torch.float32
    X = (torch.randn(T, d, generator=g, device=DEV) * scale).to(dt)
    W = (torch.randn(d, V, generator=g, device=DEV) * d ** -0.5).to(dt)
    return X, W


def check_topk(idx, lp, lse, X, W, k):
    ridx, rlp, rlse, logp = O.cache_topk(f64(X), f64(W), k)
    idx, lp = idx.cpu().numpy().astype(np.int64), f64(lp)
    assert np.abs(f64(lse) - rlse).max() <= LOGP_ATOL
    T, V = logp.shape
    assert idx.min() >= 0 and idx.max() < V
    srt = -np.sort(-logp, axis=1)
    exact = 0
    for t in range(T):
        assert len(set(idx[t])) == k                                          # distinct
        assert np.abs(lp[t] - logp[t, idx[t]]).max() <= LOGP_ATOL            # the scores are the chosen columns' log-probs
        assert logp[t, idx[t]].min() >= srt[t, k - 1] - 2 * ZTOL             # a valid top-k set
        assert np.all(np.diff(logp[t, idx[t]]) <= 2 * ZTOL)                  # descending
        gaps = -np.diff(srt[t, : min(k + 1, V)])
        if gaps.size == 0 or gaps.min() > 4 * ZTOL:                          # the fp64 decision has a margin: exact
            assert np.array_equal(idx[t], ridx[t])
        exact += int(np.array_equal(idx[t], ridx[t]))
    return exact / T


@pytest.mark.parametrize("dtype,T,d,V,k,layout", [
    ("fp32", 256, 256, 4096, 8, "dv"), ("bf16", 700, 320, 2056, 16, "dv"), ("bf16", 700, 320, 2056, 64, "vd"),
    ("bf16", 300, 128, 8200, 1, "dv"), ("bf16", 1024, 1024, 32768, 16, "dv"), ("bf16", 520, 512, 32768, 64, "vd")])
def test_cache_topk(handle, dtype, T, d, V, k, layout):
    X, W = inputs(dtype, T, d, V, 1)
    Wl = W if layout == "dv" else W.t().contiguous().t()
    idx, lp, lse = handle.cache_topk(X, Wl, k)
    torch.cuda.synchronize()
    assert check_topk(idx, lp, lse, X, W, k) > 0.9


def test_cache_topk_ties_and_peaked_rows(handle):
    """Exactly tied logits (duplicated W columns) resolve to the lowest index; peaked rows (hidden x4) still select right."""
    X, W = inputs("bf16", 260, 256, 4104, 2, scale=4.0)
    W[:, 4000] = W[:, 7]; W[:, 300] = W[:, 7]; W[:, 2049] = W[:, 2048]
    idx, lp, lse = handle.cache_topk(X, W, 32)
    torch.cuda.synchronize()
    check_topk(idx, lp, lse, X, W, 32)
    idx = idx.cpu().numpy()
    for t in range(260):
        pos = {c: np.flatnonzero(idx[t] == c) for c in (7, 300, 4000)}
        if all(p.size for p in pos.values()):
            assert pos[300][0] == pos[7][0] + 1 and pos[4000][0] == pos[7][0] + 2
        present = [c for c in (7, 300, 4000) if pos[c].size]
        assert present == [7, 300, 4000][: len(present)]                      # a lower index is never dropped first


def test_cache_topk_is_what_the_learner_consumes(handle):
    """Producer -> learner: the top-k cache built by opd_cache_topk from a teacher head feeds opd_loss_fwd_bwd."""
    cfg = dict(dtype="bf16", T=384, d=256, V=4096, k=8, K=4, sigma=0.05, mask="none")
    inp = synth.make_inputs(cfg, c=21, device=DEV, keep_teacher_rows=True)
    idx, lp, _ = handle.cache_topk(inp["hidden"], inp["W_T"], 8)
    torch.cuda.synchronize()
    r = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lp, None, inp["mask"], O.FKL_TOPK, 8, flags=32)
    ref = O.opd_oracle(f64(inp["hidden"]), f64(inp["W"]), f64(inp["topk_idx"]), f64(inp["topk_logq"]), None, f64(inp["mask"]),
                       O.FKL_TOPK, 8, want_grads=False)
    assert abs(r["loss"].item() - ref["loss"]) <= 2e-3 * abs(ref["loss"])


def check_samples(idx, lp, lse, X, W, u):
    ridx, rlp, rlse, cdf = O.cache_sample(f64(X), f64(W), f64(u))
    idx, lp, u64 = idx.cpu().numpy().astype(np.int64), f64(lp), f64(u)
    T, V = cdf.shape
    assert idx.min() >= 0 and idx.max() < V
    assert np.abs(f64(lse) - rlse).max() <= LOGP_ATOL
    logp = np.log(np.diff(np.concatenate([np.zeros((T, 1)), cdf], 1), axis=1))
    assert np.abs(lp - np.take_along_axis(logp, idx, 1)).max() <= LOGP_ATOL
    hi = np.take_along_axis(cdf, idx, 1)
    lo = np.where(idx > 0, np.take_along_axis(cdf, np.maximum(idx - 1, 0), 1), 0.0)
    assert np.all(u64 <= hi + CDF_TOL) and np.all(u64 >= lo - CDF_TOL)        # u falls on the chosen index's CDF interval
    return float((idx == ridx).mean())


@pytest.mark.parametrize("dtype,T,d,V,K,layout", [
    ("fp32", 256, 256, 4096, 4, "dv"), ("bf16", 700, 320, 2056, 5, "vd"), ("bf16", 300, 128, 8200, 64, "dv"),
    ("bf16", 1024, 1024, 32768, 16, "dv"), ("bf16", 260, 256, 151936, 8, "dv")])
def test_cache_sample(handle, dtype, T, d, V, K, layout):
    X, W = inputs(dtype, T, d, V, 3)
    u = torch.rand(T, K, generator=torch.Generator(device=DEV).manual_seed(5), device=DEV)
    u[0, 0] = 0.0; u[1, :] = 0.5; u[2, K - 1] = 1.0 - 2.0 ** -24                # edges, duplicates, the last index
    Wl = W if layout == "dv" else W.t().contiguous().t()
    idx, lp, lse = handle.cache_sample(X, Wl, u)
    torch.cuda.synchronize()
    # exact agreement is limited by the fp32 CDF resolution (~1e-7..1e-6) against the width 1/V of an index's interval
    assert check_samples(idx, lp, lse, X, W, u) > (0.995 if V <= 32768 else 0.97)
    assert torch.equal(idx[1], idx[1, :1].expand(K))


def test_cache_sample_frequencies_and_learner_roundtrip(handle):
    """Many draws of one peaked row reproduce its probabilities (chi-square); the sampled cache with its own log-probs as
    log p_old makes rho == 1 in the learner (on-policy)."""
    X, W = inputs("bf16", 256, 256, 4096, 4, scale=3.0)
    X[:] = X[0]
    u = torch.rand(256, 64, generator=torch.Generator(device=DEV).manual_seed(6), device=DEV)
    idx, lp, lse = handle.cache_sample(X, W, u)
    torch.cuda.synchronize()
    p = np.exp(O.cache_topk(f64(X[:1]), f64(W), 4096)[3][0])
    counts = np.bincount(idx.cpu().numpy().ravel(), minlength=4096).astype(np.float64)
    n = counts.sum()
    big = p * n >= 5
    chi2 = (((counts[big] - p[big] * n) ** 2) / (p[big] * n)).sum() + (counts[~big].sum() - p[~big].sum() * n) ** 2 / max(p[~big].sum() * n, 1e-9)
    dof = big.sum()
    assert chi2 < dof + 6 * np.sqrt(2 * dof)
    from paper_2606_24143_b200 import opd
    rho = torch.zeros(256, 64, device=DEV)
    handle.set_diagnostics(rho, None)
    try:
        handle.loss_fwd_bwd(X, W, idx, lp - 0.3, lp, torch.ones(256, dtype=torch.uint8, device=DEV), opd.RKL_MC, 64, flags=opd.F_FWD_ONLY)
        torch.cuda.synchronize()
    finally:
        handle.set_diagnostics(None, None)
    assert (rho - 1).abs().max().item() <= 2e-4


def test_producers_skip_masked_rows(handle):
    """mask argument of the producers: padding rows (all-zero hidden states: all V logits tie, which overflows the
    candidate list of opd_cache_topk) are not scored when masked and fail the batch when they are not; the scored rows
    give exactly what the unmasked call gives for them; rows with mask 0 are left unwritten."""
    from paper_2606_24143_b200 import opd
    T, d, V, k, K = 520, 256, 8200, 8, 6
    X, W = inputs("bf16", T, d, V, 31)
    base_idx, base_lp, base_lse = handle.cache_topk(X, W, k)
    u = torch.rand(T, K, generator=torch.Generator(device=DEV).manual_seed(5), device=DEV)
    sbase_idx, sbase_lp, _ = handle.cache_sample(X, W, u)
    torch.cuda.synchronize()
    mask = torch.ones(T, dtype=torch.uint8, device=DEV)
    dead = torch.tensor([0, 7, 255, 256, 300, T - 1], device=DEV)
    mask[dead] = 0
    Xp = X.clone(); Xp[dead] = 0                        # padding rows
    with pytest.raises(opd.OpdError) as e:
        handle.cache_topk(Xp, W, k)
    assert e.value.status == opd.ERR_WORKSPACE
    idx, lp, lse = handle.cache_topk(Xp, W, k, mask=mask)
    sidx, slp, slse = handle.cache_sample(Xp, W, u, mask=mask != 0)
    torch.cuda.synchronize()
    live = mask != 0
    assert torch.equal(idx[live], base_idx[live]) and torch.equal(lp[live], base_lp[live]) and torch.equal(lse[live], base_lse[live])
    assert torch.equal(sidx[live], sbase_idx[live]) and torch.equal(slp[live], sbase_lp[live]) and torch.equal(slse[live], base_lse[live])
    assert (idx[dead] == -1).all() and torch.isinf(lp[dead]).all() and (lse[dead] == 0).all() and (sidx[dead] == -1).all()
    none = handle.cache_topk(Xp, W, k, mask=torch.zeros_like(mask))
    torch.cuda.synchronize()
    assert (none[0] == -1).all()

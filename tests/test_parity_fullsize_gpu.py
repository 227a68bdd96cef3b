"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The fp64 oracle cannot materialise T x V at these sizes, so (i) outputs the oracle can compute one by
one — lse, per-token loss, student log-probs and whole grad_hidden rows of sampled tokens — are compared
directly, and (ii) grad_W is checked through properties that hold at any size:
   sum_v grad_W[k,v] = 0                       (softmax shift invariance, pin P10)
   sum_v W[k,v] grad_W[k,v] = sum_t x[t,k] grad_hidden[t,k]   for every k   (both equal <z, G> split by k)
plus (iii) a few-live-token variant of the 1.7B-class shape where the oracle computes grad_W in full, and (iv) grad_W element by
element on >= 256 vocabulary columns at the full T / d / V of C3, C4 and C5 (oracle.grad_W_columns: every live token contributes to
every column, so the oracle runs one fp64 forward over all live tokens; C3 keeps its own variable-length mask, C4 runs with all
32 768 tokens live and C5 with 32 768 of its 65 536, so that at least 8 token super-tiles reduce into every grad_W panel as in the
timed configuration; these two are marked `slow`: the oracle needs minutes of host time).  C4's staleness sweep (sigma = 0 / 0.1)
and the surrogate flags are covered on sampled rows and on grad_W columns of a thinned mask."""
import numpy as np
import pytest
import torch

from oracle import opd_oracle as O
from gen import synth
from tests._util import GRAD_TOL, LOGP_ATOL, LOSS_RTOL, check_grad, compare_all, f64, oracle_for, pick

pytestmark = pytest.mark.gpu
DEV = "cuda"


@pytest.fixture(scope="module")
def handle():
    from paper_2606_24143_b200 import opd
    return opd.Handle(0)


def _surrogate(flags):
    """OPD_F_SUR_CLIP (64) / OPD_F_SUR_A_OLD (128) -> the oracle's surrogate code (Eq.(6),(7) PAPER.md:132-141)."""
    return {0: O.SUR_THETA_NOCLIP, 64: O.SUR_THETA_CLIP, 128: O.SUR_OLD_NOCLIP, 192: O.SUR_OLD_CLIP}[flags & 192]


def sampled_check(handle, cfg, c, mode, n_rows=12, layout="dv", sigma=None, flags=0, rho_is_one=False):
    """sigma: staleness of the rollout policy (None = the config's); flags: surrogate flags; rho_is_one: the cache was scored by
    the current weights (sigma = 0), so every importance ratio the kernel forms must be 1 to 1e-4 (checked on ALL live slots
    through opd_set_diagnostics, not on a sample)."""
    inp = synth.make_inputs(cfg, c=c, device=DEV, sigma=sigma)
    if layout == "vd":                                       # the same logical [d,V] matrix stored [V,d] like lm_head.weight
        inp["W"] = inp["W"].t().contiguous().t()
    idx, lam, old, kk = pick(inp, cfg, mode)
    rho = torch.full(tuple(idx.shape), float("nan"), device=DEV) if rho_is_one else None
    if rho is not None:
        handle.set_diagnostics(rho_out=rho)
    try:
        r = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, flags=flags, want_lse=True,
                                want_student_logp=True)
        torch.cuda.synchronize()
    finally:
        if rho is not None:
            handle.set_diagnostics(None, None)
    if rho is not None:
        lv = rho[inp["mask"] != 0]
        assert not torch.isnan(lv).any() and float((lv - 1.0).abs().max()) <= 1e-4
    mask = f64(inp["mask"])
    live = np.flatnonzero(mask)
    rng = np.random.default_rng(c)
    rows = np.sort(np.concatenate([live[:2], rng.choice(live, n_rows - 4, replace=False), live[-2:]]))
    W = f64(inp["W"])
    sel = torch.as_tensor(rows, device=DEV)
    sub = dict(hidden=inp["hidden"][sel], W=inp["W"], mask=inp["mask"][sel])
    # the oracle on the sampled rows only, with the normaliser of the whole call
    ref = O.opd_oracle(f64(sub["hidden"]), W, f64(idx[sel]), f64(lam[sel]), f64(old[sel]) if old is not None else None,
                       f64(sub["mask"]), mode, kk, norm_override=float(live.size), want_grad_W=False, surrogate=_surrogate(flags))
    assert np.abs(f64(r["lse"][sel]) - ref["lse"]).max() <= LOGP_ATOL
    a, b = f64(r["student_logp"][sel]), ref["student_logp"]
    used = ~np.isnan(b)
    assert np.abs(a[used] - b[used]).max() <= LOGP_ATOL
    assert np.abs(f64(r["per_token_kl"][sel]) - ref["per_token_kl"]).max() <= LOSS_RTOL * np.abs(ref["per_token_kl"]).max()
    gh = r["grad_hidden"]
    check_grad(f64(gh[sel]), ref["grad_hidden"], "bf16", "grad_hidden rows")
    assert abs(r["loss"].item() - r["per_token_kl"].double().sum().item() / live.size) <= 1e-5 * max(1.0, abs(r["loss"].item()))
    if (mask == 0).any():
        dead = torch.as_tensor(np.flatnonzero(mask == 0), device=DEV)
        assert not gh[dead].any() and not r["per_token_kl"][dead].any()
    # grad_W properties (fp64 reductions of the CUDA outputs, done with torch on the GPU: test infrastructure)
    gw = r["grad_W"]
    gmax = gw.abs().max().item()
    colsum = gw.double().sum(dim=1)
    V = gw.shape[1]
    # every row of G sums to 0 up to the bf16 rounding of its entries (relative 2^-9 each): sum_v grad_W[k,v] is a random walk
    # over the live tokens of those per-row residuals, about 2^-9 sqrt(n_live * C) |x| |beta| / N against a largest entry of a few
    # |x| |beta| / N, so a bound of 1e-2 gmax sqrt(n_live) leaves a factor of about 4 (the element-wise column checks below
    # are the primary grad_W test)
    assert colsum.abs().max().item() <= 1e-2 * gmax * np.sqrt(live.size)
    lhs = (inp["W"].double() * gw.double()).sum(dim=1)
    rhs = (inp["hidden"].double() * gh.double()).sum(dim=0)
    assert (lhs - rhs).abs().max().item() <= 2e-2 * max(lhs.abs().max().item(), 1e-30)
    # a second call at full size gives the same bits: the dependency counters fix the order of every fp32 reduction whatever CTA
    # pair claims a tile (a race between a tile's stores and its publication would show up here first)
    keep = (r["loss"].clone(), gh.clone(), gw.clone())
    del r, gh, gw
    r2 = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, flags=flags)
    torch.cuda.synchronize()
    assert torch.equal(keep[0], r2["loss"]) and torch.equal(keep[1], r2["grad_hidden"]) and torch.equal(keep[2], r2["grad_W"])


def test_C3_shape_sampled(handle):
    sampled_check(handle, synth.CONFIGS[3], 3, O.RKL_MC)
    sampled_check(handle, synth.CONFIGS[3], 3, O.FKL_TOPK)


def test_C3_shape_sampled_vd_storage(handle):
    """W stored [V,d] (other TMA boxes / UMMA majorness in all three contractions), at the 1.7B-class shape."""
    sampled_check(handle, synth.CONFIGS[3], 3, O.RKL_MC, layout="vd")


def test_C4_shape_sampled(handle):
    sampled_check(handle, synth.CONFIGS[4], 4, O.RKL_MC)


def test_C4_staleness_sweep_is_parity_tested(handle):
    """BASELINE.json configs[3]: "staleness sweep with W_old perturbation 0.0/0.02/0.1" (0.02 is test_C4_shape_sampled).
    sigma = 0: the cache holds the current student's own log-probs, so rho = 1 on every live slot (to 1e-4) and the sampled rows
    match the oracle; sigma = 0.1 (p99 of rho about 1.26: the clip bites) with the clipped A_old surrogate, sampled rows."""
    sampled_check(handle, synth.CONFIGS[4], 4, O.RKL_MC, sigma=0.0, rho_is_one=True)
    sampled_check(handle, synth.CONFIGS[4], 4, O.RKL_MC, sigma=0.1, flags=192)


def test_C5_shape_sampled_mixed(handle):
    sampled_check(handle, synth.CONFIGS[5], 5, O.MIXED)


def test_C3_shape_few_live_tokens_full_oracle(handle):
    """d=2048, V=151936 with 160 live tokens scattered over T=16384: every output against the full oracle."""
    cfg = dict(synth.CONFIGS[3])
    inp = synth.make_inputs(cfg, c=3, device=DEV)
    m = torch.zeros_like(inp["mask"])
    sel = torch.randperm(cfg["T"], generator=torch.Generator().manual_seed(5))[:160].to(DEV)
    m[sel] = 1
    inp["mask"] = m
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    r = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, m, O.RKL_MC, kk, want_lse=True, want_student_logp=True)
    torch.cuda.synchronize()
    compare_all(r, oracle_for(inp, idx, lam, old, O.RKL_MC, kk, chunk=32), f64(m), "bf16")


def test_C4_shape_sparse_reverse_kl_sampled(handle):
    """OPD_RKL_TOPK (stale student support, sparse backward) at the C4 shape on sampled rows."""
    sampled_check(handle, synth.CONFIGS[4], 4, O.RKL_TOPK)


def test_producers_at_C3_shape_sampled_rows(handle):
    """opd_cache_topk / opd_cache_sample at T=16384, d=2048, V=151936 in the launch configuration bench.py --op times:
    validity of the sampled rows against the fp64 oracle (each row needs only its own logits)."""
    cfg = synth.CONFIGS[3]
    inp = synth.make_inputs(cfg, c=3, device=DEV)
    X, W = inp["hidden"], inp["W"]
    T, V = cfg["T"], cfg["V"]
    k = cfg["k"]
    idx, lp, lse = handle.cache_topk(X, W, k)
    u = torch.rand(T, cfg["K"], generator=torch.Generator(device=DEV).manual_seed(9), device=DEV)
    sidx, slp, slse = handle.cache_sample(X, W, u)
    torch.cuda.synchronize()
    assert torch.equal(lse, slse)
    assert int(idx.min()) >= 0 and int(idx.max()) < V and int(sidx.min()) >= 0 and int(sidx.max()) < V
    rows = np.sort(np.random.default_rng(3).choice(T, 16, replace=False))
    sel = torch.as_tensor(rows, device=DEV)
    Xs, Wd = f64(X[sel]), f64(W)
    ridx, rlp, rlse, logp = O.cache_topk(Xs, Wd, k)
    gi, gl = idx[sel].cpu().numpy().astype(np.int64), f64(lp[sel])
    assert np.abs(f64(lse[sel]) - rlse).max() <= LOGP_ATOL
    srt = -np.sort(-logp, axis=1)
    for r in range(len(rows)):
        assert len(set(gi[r])) == k
        assert np.abs(gl[r] - logp[r, gi[r]]).max() <= LOGP_ATOL
        assert logp[r, gi[r]].min() >= srt[r, k - 1] - 2e-4 and np.all(np.diff(logp[r, gi[r]]) <= 2e-4)
    assert np.mean([np.array_equal(gi[r], ridx[r]) for r in range(len(rows))]) >= 0.75
    _, _, _, cdf = O.cache_sample(Xs, Wd, f64(u[sel]))
    si, u64 = sidx[sel].cpu().numpy().astype(np.int64), f64(u[sel])
    hi = np.take_along_axis(cdf, si, 1)
    lo = np.where(si > 0, np.take_along_axis(cdf, np.maximum(si - 1, 0), 1), 0.0)
    assert np.all(u64 <= hi + 2e-5) and np.all(u64 >= lo - 2e-5)
    assert np.abs(f64(slp[sel]) - np.take_along_axis(logp, si, 1)).max() <= LOGP_ATOL


def _columns_for(idx, live, V, rng, n_tok=16, n_rand=96):
    """>= 256 vocabulary columns: every cached column of n_tok random live tokens (where the sparse beta terms land), random
    columns, and the last, partial vocabulary tile (V = 151936 = 593 * 256 + 128)."""
    toks = rng.choice(live, n_tok, replace=False)
    cached = np.unique(f64(idx[torch.as_tensor(toks, device=idx.device)]).astype(np.int64).ravel())
    cached = cached[(cached >= 0) & (cached < V)][:160]
    tail = np.arange(V - V % 256 if V % 256 else V - 256, V)
    return np.unique(np.concatenate([cached, rng.choice(V, n_rand, replace=False), tail, [0, 255, 256, 4095, 4096]]))


def grad_W_column_check(handle, cfg, c, mode, n_live_target=None, layout="dv", flags=0, sigma=None):
    inp = synth.make_inputs(cfg, c=c, device=DEV, sigma=sigma)
    T, V = cfg["T"], cfg["V"]
    if n_live_target is not None:        # scattered subset of the live tokens (the mode codes of OPD_MIXED are kept)
        live0 = torch.nonzero(inp["mask"] != 0).flatten()
        keep = live0[torch.randperm(live0.numel(), generator=torch.Generator().manual_seed(c))[:n_live_target].to(DEV)]
        m = torch.zeros_like(inp["mask"])
        m[keep] = inp["mask"][keep]
        inp["mask"] = m
    idx, lam, old, kk = pick(inp, cfg, mode)
    W = inp["W"] if layout == "dv" else inp["W"].t().contiguous().t()
    r = handle.loss_fwd_bwd(inp["hidden"], W, idx, lam, old, inp["mask"], mode, kk, flags=flags)
    torch.cuda.synchronize()
    st = handle.launch_stats()
    mask = f64(inp["mask"])
    live = np.flatnonzero(mask)
    assert live.size > st["super_rows"], "the check must span more than one token super-tile"
    cols = _columns_for(idx, live, V, np.random.default_rng(100 + c))
    assert cols.size >= 256
    ref = O.grad_W_columns(f64(inp["hidden"]), f64(inp["W"]), f64(idx), f64(lam), f64(old) if old is not None else None, mask,
                           mode, kk, cols, surrogate=_surrogate(flags))
    got = f64(r["grad_W"][:, torch.as_tensor(cols, device=DEV)])
    # the bar is relative to the largest entry of the compared columns (they hold the cached columns, where grad_W peaks)
    check_grad(got, ref, "bf16", f"grad_W[:, {cols.size} columns] at {cfg['name']}")
    # per-column: no single column may hide behind the global maximum by more than 4x its own scale
    col_scale = np.maximum(np.abs(ref).max(axis=0), 1e-3 * np.abs(ref).max())
    assert (np.abs(got - ref).max(axis=0) <= 4 * GRAD_TOL["bf16"] * col_scale).all()
    return r, inp


def test_C3_grad_W_columns_full_mask(handle):
    """C3 (T=16384, d=2048, V=151936, variable-length mask, ~9.2k live tokens): grad_W columns element by element, both modes."""
    grad_W_column_check(handle, synth.CONFIGS[3], 3, O.RKL_MC)
    grad_W_column_check(handle, synth.CONFIGS[3], 3, O.FKL_TOPK, layout="vd")


def test_C4_grad_W_columns_surrogate_thinned(handle):
    """C4 (T=32768, d=4096, V=151936) with sigma = 0.1 and the clipped A_old surrogate (flags 192): 6144 scattered live tokens
    (two token super-tiles, all vocabulary super-tiles), grad_W columns element by element."""
    grad_W_column_check(handle, synth.CONFIGS[4], 4, O.RKL_MC, n_live_target=6144, flags=192, sigma=0.1)


@pytest.mark.slow
def test_C4_grad_W_columns_all_tokens_live(handle):
    """The configuration bench.py times, unthinned: all 32 768 tokens live, so each grad_W panel is the sum of the 8 token
    super-tiles' reduce-add passes.  >= 256 columns (cached columns, random ones, the last partial vocabulary tile) element by
    element.  The oracle's fp64 forward over 32 768 x 151 936 logits takes about two minutes of host time."""
    r, inp = grad_W_column_check(handle, synth.CONFIGS[4], 4, O.RKL_MC)
    assert int((inp["mask"] != 0).sum()) == 32768 and 32768 // handle.launch_stats()["super_rows"] >= 8


@pytest.mark.slow
def test_C5_grad_W_columns_mixed(handle):
    """C5 (T=65536, d=2560, V=151936, mixed FKL k=64 / MC K=8 rows): 32 768 scattered live tokens over all 16 token super-tiles
    (>= 8 of them reduce into each panel)."""
    r, inp = grad_W_column_check(handle, synth.CONFIGS[5], 5, O.MIXED, n_live_target=32768)
    assert 65536 // handle.launch_stats()["super_rows"] >= 8

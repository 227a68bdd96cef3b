"""GPU parity: the CUDA path (through the C ABI binding) against the fp64 oracle, element by element,
on the same seeded inputs.  Run with `-m gpu` on a B200."""
import os

import numpy as np
import pytest
import torch

from oracle import opd_oracle as O
from gen import synth
from tests._util import GRAD_TOL, LOGP_ATOL, check_grad, check_loss, compare_all, f64, oracle_for, pick

pytestmark = pytest.mark.gpu
DEV = "cuda"


@pytest.fixture(scope="module")
def opd():
    from paper_2606_24143_b200 import opd as m
    return m


@pytest.fixture(scope="module")
def handle(opd):
    return opd.Handle(0)


def run(handle, inp, idx, lam, old, mode, kk, flags=0, layout="dv", **kw):
    W = inp["W"] if layout == "dv" else inp["W"].t().contiguous().t()     # same logical [d,V], [V,d] storage
    r = handle.loss_fwd_bwd(inp["hidden"], W, idx, lam, old, inp["mask"], mode, kk, flags=flags, want_lse=True,
                            want_student_logp=True, **kw)
    torch.cuda.synchronize()
    return r


# ------------------------------------------------------------------------------------------------
def test_gemm_core_all_operand_layouts(handle):
    """The tcgen05 core against torch fp32 matmul for K-major / MN-major A and B, with ragged M, N, K."""
    torch.manual_seed(1)
    for (M, N, K) in [(128, 256, 64), (200, 304, 200), (1000, 1000, 520)]:
        A = torch.randn(M, K, device=DEV).bfloat16()
        B = torch.randn(N, K, device=DEV).bfloat16()
        ref = A.double() @ B.double().t()
        for amn in (False, True):
            for bmn in (False, True):
                D = handle.debug_gemm(A.t().contiguous() if amn else A, B.t().contiguous() if bmn else B, amn, bmn)
                torch.cuda.synchronize()
                assert (D.double() - ref).abs().max() <= 2e-5 * ref.abs().max()


@pytest.mark.parametrize("dtype", ["bf16", "fp32"])
@pytest.mark.parametrize("layout", ["dv", "vd"])
def test_gathers_are_bit_exact(handle, dtype, layout):
    """north_star 'cache gathers bit-exact' (reading Q12): the gathered value is bit-identical to the
    fp32 logit the same kernel held at (t, a_tj); duplicates in a row give identical values; unsorted caller order."""
    torch.manual_seed(2)
    T, d, V, C = 300, 256, 4104, 8
    dt = torch.bfloat16 if dtype == "bf16" else torch.float32
    X = torch.randn(T, d, device=DEV).to(dt)
    W = (torch.randn(d, V, device=DEV) / 16).to(dt)
    idx = torch.randint(0, V, (T, C), device=DEV, dtype=torch.int32)
    idx[:, 5] = idx[:, 1]
    idx[0] = torch.tensor([V - 1, 0, 255, 256, 257, 0, V - 8, 4095], dtype=torch.int32)
    Wl = W if layout == "dv" else W.t().contiguous().t()
    logits, gathered = handle.debug_logits(X, Wl, idx)
    torch.cuda.synchronize()
    assert torch.equal(gathered, torch.gather(logits, 1, idx.long()))
    assert torch.equal(gathered[:, 5], gathered[:, 1])
    z = f64(X) @ f64(W)
    assert np.abs(f64(logits) - z).max() <= (2e-5 if dtype == "bf16" else 5e-5)


@pytest.mark.parametrize("mode,flags,layout", [
    (O.FKL_TOPK, 0, "dv"), (O.FKL_TOPK, 0, "vd"), (O.RKL_MC, 0, "dv"), (O.RKL_MC, 0, "vd"),
    (O.FKL_TOPK, O.F_RENORM_STUDENT, "dv"), (O.FKL_TOPK, O.F_NO_RENORM_TEACHER, "dv"),
    (O.FKL_TOPK, O.F_NO_RENORM_TEACHER | O.F_RENORM_STUDENT, "vd"),
    (O.RKL_MC, 64, "dv"), (O.RKL_MC, 128, "dv"), (O.RKL_MC, 64 | 128, "dv"), (O.RKL_TOPK, 0, "dv"), (O.RKL_TOPK, 0, "vd")])
def test_C1_fp32(handle, mode, flags, layout):
    """BASELINE.json configs[0]: fp32, T=256, d=256, V=4096, k=8 / K=4, sigma=0.05, 10% masked."""
    cfg = synth.CONFIGS[1]
    inp = synth.make_inputs(cfg, c=1, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, mode)
    r = run(handle, inp, idx, lam, old, mode, kk, flags, layout)
    compare_all(r, oracle_for(inp, idx, lam, old, mode, kk, flags), f64(inp["mask"]), "fp32")


@pytest.mark.parametrize("mode", [O.FKL_TOPK, O.RKL_MC, O.RKL_TOPK])
def test_C2_bf16(handle, mode):
    """BASELINE.json configs[1]: bf16, T=4096, d=1024, V=32768, k=16 / K=4, sigma=0.02 (full oracle)."""
    cfg = synth.CONFIGS[2]
    inp = synth.make_inputs(cfg, c=2, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, mode)
    r = run(handle, inp, idx, lam, old, mode, kk)
    compare_all(r, oracle_for(inp, idx, lam, old, mode, kk), f64(inp["mask"]), "bf16")


RAGGED = dict(dtype="bf16", T=700, d=320, V=2056, k=8, K=5, sigma=0.05, mask="random10")


@pytest.mark.parametrize("dtype", ["bf16", "fp32"])
@pytest.mark.parametrize("mode", [O.FKL_TOPK, O.RKL_MC, O.MIXED, O.RKL_TOPK])
@pytest.mark.parametrize("tiles", [None, (256, 512)])
def test_ragged_shapes_and_super_tiles(handle, dtype, mode, tiles, monkeypatch):
    """T, V not multiples of the tile sizes, d not a multiple of 256; several backward super-tiles in both
    directions (OPD_TB / OPD_VB shrink them) must give the same result as one."""
    if tiles:
        monkeypatch.setenv("OPD_TB", str(tiles[0]))
        monkeypatch.setenv("OPD_VB", str(tiles[1]))
    cfg = dict(RAGGED, dtype=dtype)
    inp = synth.make_inputs(cfg, c=7, device=DEV)
    if mode == O.MIXED:
        m = inp["mask"].clone()
        m[(torch.arange(cfg["T"], device=DEV) % 3 == 0) & (m != 0)] = 2
        inp["mask"] = m
    idx, lam, old, kk = pick(inp, cfg, mode)
    r = run(handle, inp, idx, lam, old, mode, kk)
    compare_all(r, oracle_for(inp, idx, lam, old, mode, kk), f64(inp["mask"]), dtype)
    if tiles:
        assert handle.launch_stats()["super_rows"] == tiles[0]


@pytest.mark.parametrize("dtype", ["bf16", "fp32"])
@pytest.mark.parametrize("mode,flags", [(O.RKL_TOPK, 0), (O.FKL_TOPK, O.F_RENORM_STUDENT)])
@pytest.mark.parametrize("layout", ["dv", "vd"])
def test_sparse_backward_hot_columns(handle, dtype, mode, flags, layout):
    """Skewed supports (gen/synth hot_columns): three columns sit in the support of (almost) every row, so their runs of sorted
    cache entries are ~1350 long and span several of the sparse backward's 256-entry segments (summed by k_sparse_gw_seg and added
    in segment order); d = 1280 needs two k-chunks.  Element-wise against the oracle, and bitwise equal on a second call."""
    cfg = dict(dtype=dtype, T=1500, d=1280, V=2056, k=8, K=4, sigma=0.05, mask="random10", hot_columns=3)
    inp = synth.make_inputs(cfg, c=23, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, mode)
    live = inp["mask"] != 0
    assert int((idx[live] == 7).sum()) > 4 * 256                    # the hot column's run really spans several segments
    r = run(handle, inp, idx, lam, old, mode, kk, flags, layout)
    compare_all(r, oracle_for(inp, idx, lam, old, mode, kk, flags), f64(inp["mask"]), dtype)
    r2 = run(handle, inp, idx, lam, old, mode, kk, flags, layout)
    assert torch.equal(r["grad_W"], r2["grad_W"]) and torch.equal(r["grad_hidden"], r2["grad_hidden"])
    W = inp["W"] if layout == "dv" else inp["W"].t().contiguous().t()
    gw = torch.empty_strided(tuple(W.shape), W.stride(), dtype=torch.float32, device=DEV).fill_(1.0)
    r3 = handle.loss_fwd_bwd(inp["hidden"], W, idx, lam, old, inp["mask"], mode, kk, flags=flags | 4, grad_W=gw)   # OPD_F_GRADW_ACCUM: added onto 1.0
    torch.cuda.synchronize()
    assert (r3["grad_W"] - 1.0 - r["grad_W"]).abs().max() <= 1e-6 * max(1.0, float(r["grad_W"].abs().max()))


STRESS = {
    "peaked": dict(hidden_scale=4.0, sigma=0.05),                   # a few columns hold the mass, most exponentials are tiny
    "monotone": dict(order="monotone", sigma=0.05),                 # the row maximum keeps moving to later vocabulary tiles
    "peaked_monotone_stale": dict(hidden_scale=3.0, order="monotone", sigma=0.3),   # + heavy tails of rho = p_theta / p_old
}


@pytest.mark.parametrize("variant", sorted(STRESS))
@pytest.mark.parametrize("dtype", ["bf16", "fp32"])
@pytest.mark.parametrize("mode", [O.FKL_TOPK, O.RKL_MC])
def test_stress_variants(handle, variant, dtype, mode):
    """SURVEY 8(d) stress inputs: peaked rows, monotonically growing column norms (online-max rescaling in every tile of the
    forward, exponents far below zero in the re-formed softmax tiles), stale caches with large importance ratios."""
    cfg = dict(RAGGED, dtype=dtype, T=520, V=4360, **STRESS[variant])
    inp = synth.make_inputs(cfg, c=11, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, mode)
    r = run(handle, inp, idx, lam, old, mode, kk)
    ref = oracle_for(inp, idx, lam, old, mode, kk)
    if variant == "peaked_monotone_stale" and mode == O.RKL_MC:
        rho = np.exp(ref["student_logp"][:, :kk] - f64(old))
        assert np.nanmax(rho[f64(inp["mask"]) != 0]) > 3.0           # the tail is really there
    compare_all(r, ref, f64(inp["mask"]), dtype)


def stale_clip_inputs(dtype, mode):
    """A stale cache on which the PPO clip is active on both sides with advantages of both signs, without the extreme ratios
    that would let a few slots dominate the max-abs bar: the rollout-time log-probs are placed at fixed distances from the
    current student's (rho = exp(shift), shift in {+-0.9, +-0.45, +0.05, -0.07}: 2.46, 0.41, 1.57, 0.64, 1.05, 0.93 -- none
    near a clip edge, so fp64 and the kernel's fp32 take the same branch), and the teacher scores around both
    (lam = (ell + old)/2 + 0.8 N(0,1), seeded).  `ell` comes from the oracle's forward.  Returns the inputs, the caches, a
    boolean [T,K] array of the live Monte-Carlo slots and ell on them."""
    cfg = dict(RAGGED, dtype=dtype, T=520, V=4360, K=8)
    inp = synth.make_inputs(cfg, c=11, device=DEV)
    if mode == O.MIXED:
        m = inp["mask"].clone()
        m[(torch.arange(cfg["T"], device=DEV) % 3 != 0) & (m != 0)] = 2
        inp["mask"] = m
    idx, lam, old, kk = pick(inp, cfg, mode)
    Km = kk >> 16 if mode == O.MIXED else kk
    mk = f64(inp["mask"])
    slots = np.zeros(tuple(idx.shape), dtype=bool)
    slots[(mk == 2) if mode == O.MIXED else (mk != 0), :Km] = True
    ell = oracle_for(inp, idx, lam, old, mode, kk, want_grads=False)["student_logp"]
    rng = np.random.default_rng(77)
    shift = rng.choice(np.array([0.9, -0.9, 0.45, -0.45, 0.05, -0.07]), size=slots.shape)
    old64 = np.where(slots, ell - shift, f64(old))
    lam64 = np.where(slots, 0.5 * (ell + old64) + 0.8 * rng.normal(size=slots.shape), f64(lam))   # FKL rows keep their teacher cache
    old = torch.as_tensor(old64, dtype=torch.float32, device=DEV)
    lam = torch.as_tensor(lam64, dtype=torch.float32, device=DEV)
    return inp, idx, lam, old, kk, slots, np.where(slots, ell, np.nan)


@pytest.mark.parametrize("dtype", ["bf16", "fp32"])
@pytest.mark.parametrize("mode", [O.RKL_MC, O.MIXED])
@pytest.mark.parametrize("flags", [64, 128, 192])
def test_surrogates_reach_every_clip_corner(handle, dtype, mode, flags):
    """OPD_F_SUR_CLIP / OPD_F_SUR_A_OLD (Eq.(4); Eq.(6),(7) PAPER.md:132-141; eps = 0.2 PAPER.md:330) on inputs where
    the clip is active on both sides with advantages of both signs: before comparing, the oracle's rho and A must put at least
    8 live slots into each of the four corners (rho > 1.2 | rho < 0.8) x (A > 0 | A < 0), for the advantage the flag selects."""
    inp, idx, lam, old, kk, slots, ell = stale_clip_inputs(dtype, mode)
    rho = np.exp(ell - f64(old))
    A = (f64(lam) - f64(old)) if flags & 128 else (f64(lam) - ell)
    for hi in (True, False):
        for pos in (True, False):
            n = int((slots & ((rho > 1.2) if hi else (rho < 0.8)) & ((A > 0) if pos else (A < 0))).sum())
            assert n >= 8, (hi, pos, n)
    assert np.nanmin(np.abs(np.abs(rho - 1.0) - 0.2)) > 0.1                   # no slot near a clip edge
    r = run(handle, inp, idx, lam, old, mode, kk, flags)
    ref = oracle_for(inp, idx, lam, old, mode, kk, flags)
    compare_all(r, ref, f64(inp["mask"]), dtype)
    # discriminating power: the other three surrogates give gradients that differ from this one by many times the bar, so a
    # kernel that dropped the clip, clipped the wrong side or took the other advantage could not pass
    for other_flags in ({0, 64, 128, 192} - {flags}):
        other = oracle_for(inp, idx, lam, old, mode, kk, other_flags, want_grad_W=False)
        gap = np.abs(other["grad_hidden"] - ref["grad_hidden"]).max() / np.abs(ref["grad_hidden"]).max()
        assert gap > 10 * GRAD_TOL[dtype], (other_flags, gap)


def test_degenerate_cases(handle, opd):
    cfg = dict(RAGGED, T=130, k=64, K=64)
    inp = synth.make_inputs(cfg, c=8, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    # C = 64 with many duplicates (iid with replacement)
    r = run(handle, inp, idx, lam, old, O.RKL_MC, kk)
    compare_all(r, oracle_for(inp, idx, lam, old, O.RKL_MC, kk), f64(inp["mask"]), "bf16")
    # all K entries the same action == the K=1 result (pin P13 on the GPU)
    i1, l1, o1 = idx[:, :1].contiguous(), lam[:, :1].contiguous(), old[:, :1].contiguous()
    a = run(handle, inp, i1, l1, o1, O.RKL_MC, 1)
    b = run(handle, inp, i1.repeat(1, 7).contiguous(), l1.repeat(1, 7).contiguous(), o1.repeat(1, 7).contiguous(), O.RKL_MC, 7)
    assert torch.allclose(a["per_token_kl"], b["per_token_kl"], rtol=1e-5, atol=1e-6)
    # everything masked: N = 0 -> loss 0, all gradients exactly 0
    z = dict(inp, mask=torch.zeros_like(inp["mask"]))
    r = run(handle, z, idx, lam, old, O.RKL_MC, kk)
    assert r["loss"].item() == 0 and not r["grad_hidden"].any() and not r["grad_W"].any() and not r["per_token_kl"].any()
    # a single live token, and T = 1
    one = torch.zeros_like(inp["mask"]); one[77] = 1
    s = dict(inp, mask=one)
    r = run(handle, s, idx, lam, old, O.RKL_MC, kk)
    compare_all(r, oracle_for(s, idx, lam, old, O.RKL_MC, kk), f64(one), "bf16")
    t1 = dict(hidden=inp["hidden"][:1].contiguous(), W=inp["W"], mask=inp["mask"][:1] * 0 + 1)
    r = run(handle, t1, idx[:1].contiguous(), lam[:1].contiguous(), old[:1].contiguous(), O.RKL_MC, kk)
    compare_all(r, oracle_for(t1, idx[:1], lam[:1], old[:1], O.RKL_MC, kk), np.ones(1), "bf16")


def test_options_strides_and_errors(handle, opd):
    cfg = RAGGED
    inp = synth.make_inputs(cfg, c=9, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    ref = oracle_for(inp, idx, lam, old, O.RKL_MC, kk)
    T, d, V = cfg["T"], cfg["d"], cfg["V"]
    # padded row strides of hidden / caches / grads
    hp = torch.zeros(T, d + 64, device=DEV, dtype=torch.bfloat16); hp[:, :d] = inp["hidden"]
    ip = torch.full((T, kk + 3), -5, device=DEV, dtype=torch.int32); ip[:, :kk] = idx
    lp = torch.zeros(T, kk + 3, device=DEV); lp[:, :kk] = lam
    op = torch.zeros(T, kk + 3, device=DEV); op[:, :kk] = old
    ghp = torch.full((T, d + 64), 7.0, device=DEV, dtype=torch.bfloat16)
    gwp = torch.full((d, V + 8), 7.0, device=DEV)
    r = handle.loss_fwd_bwd(hp[:, :d], inp["W"], ip[:, :kk], lp[:, :kk], op[:, :kk], inp["mask"], O.RKL_MC, kk,
                            grad_hidden=ghp[:, :d], grad_W=gwp[:, :V])
    torch.cuda.synchronize()
    check_loss(r["loss"].item(), ref)
    check_grad(f64(ghp[:, :d]), ref["grad_hidden"], "bf16")
    check_grad(f64(gwp[:, :V]), ref["grad_W"], "bf16")
    assert (ghp[:, d:] == 7).all() and (gwp[:, V:] == 7).all()            # padding untouched
    # norm_override and GRADW_ACCUM (two micro-batches accumulate)
    gw = torch.zeros(d, V, device=DEV)
    for _ in range(2):
        r2 = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk, flags=opd.F_GRADW_ACCUM,
                                 norm_override=2.0 * ref["N"], grad_W=gw)
    torch.cuda.synchronize()
    assert abs(r2["loss"].item() - ref["loss"] / 2) <= 2e-3 * abs(ref["loss"])
    check_grad(f64(gw), ref["grad_W"], "bf16")
    # forward only
    r3 = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk, flags=opd.F_FWD_ONLY)
    assert r3["grad_W"] is None and abs(r3["loss"].item() - r["loss"].item()) < 1e-6
    # index validation
    bad = idx.clone(); bad[5, 0] = V
    live5 = inp["mask"][5].item() != 0
    if live5:
        with pytest.raises(opd.OpdError) as e:
            handle.loss_fwd_bwd(inp["hidden"], inp["W"], bad, lam, old, inp["mask"], O.RKL_MC, kk, flags=opd.F_VALIDATE_IDX)
        assert e.value.status == opd.ERR_BAD_INDEX
    # argument errors are reported, not crashed on
    for kwargs, code in [(dict(k_or_K=0), opd.ERR_BAD_SHAPE), (dict(k_or_K=65), opd.ERR_BAD_SHAPE), (dict(flags=1 << 20), opd.ERR_BAD_ARG)]:
        with pytest.raises(opd.OpdError) as e:
            handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC,
                                kwargs.get("k_or_K", kk), flags=kwargs.get("flags", 0))
        assert e.value.status == code
    with pytest.raises(opd.OpdError):
        handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, None, inp["mask"], O.RKL_MC, kk)
    # the host-buffer entry point gives the same numbers
    hr = handle.loss_fwd_bwd_host(inp["hidden"].cpu(), inp["W"].cpu(), idx.cpu(), lam.cpu(), old.cpu(), inp["mask"].cpu(), O.RKL_MC, kk)
    assert abs(hr["loss"].item() - r["loss"].item()) < 1e-6
    check_grad(f64(hr["grad_W"]), ref["grad_W"], "bf16")
    assert hr["h2d_bytes"] > 0 and hr["d2h_bytes"] > 0


def test_no_logits_sized_workspace(handle, opd):
    """'full logits never touch HBM' (i): no T x V sized buffer exists."""
    for c in (3, 4, 5):
        cfg = synth.CONFIGS[c]
        C = max(cfg["k"], cfg["K"])
        ws = handle.workspace_bytes(cfg["T"], cfg["d"], cfg["V"], C, opd.BF16, opd.RKL_MC, 0)
        assert ws < 0.05 * cfg["T"] * cfg["V"] * 2, (c, ws)


def test_mc_diagnostics_outputs(handle, opd):
    """opd_set_diagnostics: rho_theta per cached draw and the one-sample variance of Eq.(16) against the oracle;
    rows that are masked or not RKL_MC are left untouched / zero."""
    cfg = dict(RAGGED, K=6)
    inp = synth.make_inputs(cfg, c=11, device=DEV)
    m = inp["mask"].clone()
    m[(torch.arange(cfg["T"], device=DEV) % 2 == 0) & (m != 0)] = 2
    inp["mask"] = m
    idx, lam, old, kk = synth.mixed_cache(inp)
    rho = torch.full(idx.shape, -7.0, device=DEV)
    var1 = torch.full((cfg["T"],), -7.0, device=DEV)
    handle.set_diagnostics(rho, var1)
    try:
        handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, m, O.MIXED, kk)
        torch.cuda.synchronize()
    finally:
        handle.set_diagnostics(None, None)
    ref = oracle_for(inp, idx, lam, old, O.MIXED, kk)
    used = ~np.isnan(ref["rho"])
    got = f64(rho)
    assert np.abs(got[used] / ref["rho"][used] - 1).max() <= 2e-4
    assert np.all(got[~used] == -7.0)
    v = f64(var1)
    assert np.abs(v - ref["var1"]).max() <= 1e-3 * max(1e-30, np.abs(ref["var1"]).max())
    assert np.all(v[f64(m) != 2] == 0)


def test_seq_diagnostics_outputs(handle, opd):
    """opd_set_seq_diagnostics (Eq.(17)): per-sequence timestep averages of the m-sample and one-sample
    estimators and the fixed-path variance, against the oracle; MIXED batch (only the RKL_MC rows take part), ragged
    sequence boundaries, an empty sequence and one that holds no MC row."""
    cfg = dict(RAGGED, K=6)
    inp = synth.make_inputs(cfg, c=19, device=DEV)
    T = cfg["T"]
    m = inp["mask"].clone()
    m[(torch.arange(T, device=DEV) % 2 == 0) & (m != 0)] = 2
    m[100:140][m[100:140] == 2] = 1                       # a sequence without any MC row
    inp["mask"] = m
    idx, lam, old, kk = synth.mixed_cache(inp)
    cu = torch.tensor([0, 37, 100, 140, 140, 512, T], dtype=torch.int32, device=DEV)
    out = handle.set_seq_diagnostics(cu)
    try:
        handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, m, O.MIXED, kk)
        torch.cuda.synchronize()
    finally:
        handle.set_seq_diagnostics(None)
    ref = oracle_for(inp, idx, lam, old, O.MIXED, kk)
    K = kk >> 16
    mm, m1, vm = O.seq_diagnostics(ref["per_token_kl"], ref["first_draw"], ref["var1"], f64(m), cu.cpu().numpy(), K, mc_code=2)
    for got, want in ((out["seq_mean_m"], mm), (out["seq_mean_1"], m1), (out["seq_var_m"], vm)):
        g = f64(got)
        assert np.abs(g - want).max() <= 2e-3 * max(1e-30, np.abs(want).max())
        assert g[2] == 0 and g[3] == 0                    # no MC row / empty sequence
    # plain RKL_MC: every live row takes part
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    out = handle.set_seq_diagnostics(cu)
    try:
        handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, m, O.RKL_MC, kk)
        torch.cuda.synchronize()
    finally:
        handle.set_seq_diagnostics(None)
    ref = oracle_for(inp, idx, lam, old, O.RKL_MC, kk)
    mm, m1, vm = O.seq_diagnostics(ref["per_token_kl"], ref["first_draw"], ref["var1"], f64(m), cu.cpu().numpy(), kk)
    assert np.abs(f64(out["seq_mean_m"]) - mm).max() <= 2e-3 * np.abs(mm).max()
    assert np.abs(f64(out["seq_mean_1"]) - m1).max() <= 2e-3 * np.abs(m1).max()
    assert np.abs(f64(out["seq_var_m"]) - vm).max() <= 2e-3 * np.abs(vm).max()
    # surrogate flags would mix objectives in the three outputs (per-token values follow the surrogate, the one-sample terms do
    # not): refused on the host while the hook is on, accepted again once it is off
    handle.set_seq_diagnostics(cu)
    try:
        for fl in (opd.F_SUR_CLIP, opd.F_SUR_A_OLD, opd.F_SUR_CLIP | opd.F_SUR_A_OLD):
            with pytest.raises(opd.OpdError) as e:
                handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, m, O.RKL_MC, kk, flags=fl)
            assert e.value.status == opd.ERR_BAD_ARG and "opd_set_seq_diagnostics" in str(e.value)
    finally:
        handle.set_seq_diagnostics(None)
    handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, m, O.RKL_MC, kk, flags=opd.F_SUR_CLIP)
    torch.cuda.synchronize()


@pytest.mark.parametrize("case", ["C1", "C2", "ragged_vd", "ragged_sparse"])
def test_grad_W_bf16_output(handle, opd, case):
    """OPD_F_GRADW_BF16 (reading Q15): grad_W as a bf16 array, summed in fp32 and rounded once at the end;
    with OPD_F_GRADW_ACCUM the rounded sum of the old contents and this call; the host entry copies half the bytes back."""
    cfg = {"C1": synth.CONFIGS[1], "C2": synth.CONFIGS[2]}.get(case, RAGGED)
    c = {"C1": 1, "C2": 2}.get(case, 21)
    mode = O.RKL_TOPK if case == "ragged_sparse" else O.RKL_MC
    inp = synth.make_inputs(cfg, c=c, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, mode)
    W = inp["W"].t().contiguous().t() if case == "ragged_vd" else inp["W"]
    ref = oracle_for(inp, idx, lam, old, mode, kk)
    r = handle.loss_fwd_bwd(inp["hidden"], W, idx, lam, old, inp["mask"], mode, kk, flags=opd.F_GRADW_BF16)
    torch.cuda.synchronize()
    assert r["grad_W"].dtype == torch.bfloat16 and r["grad_W"].stride() == W.stride()
    check_loss(r["loss"].item(), ref)
    check_grad(f64(r["grad_W"]), ref["grad_W"], "bf16", "bf16 grad_W")
    check_grad(f64(r["grad_hidden"]), ref["grad_hidden"], cfg["dtype"], "grad_hidden")
    # the bf16 array is the rounding of the fp32 result of the default call (same sums, one rounding)
    r32 = handle.loss_fwd_bwd(inp["hidden"], W, idx, lam, old, inp["mask"], mode, kk)
    torch.cuda.synchronize()
    assert (r["grad_W"].float() - r32["grad_W"]).abs().max().item() <= 2.0 ** -8 * r32["grad_W"].abs().max().item()
    # accumulate: twice the gradient, rounded after the fp32 add
    gw = r["grad_W"].clone()
    handle.loss_fwd_bwd(inp["hidden"], W, idx, lam, old, inp["mask"], mode, kk, flags=opd.F_GRADW_BF16 | opd.F_GRADW_ACCUM, grad_W=gw)
    torch.cuda.synchronize()
    check_grad(f64(gw), 2.0 * ref["grad_W"], "bf16", "accumulated bf16 grad_W")
    if case == "ragged_vd":
        return
    hr = handle.loss_fwd_bwd_host(inp["hidden"].cpu(), inp["W"].cpu(), idx.cpu(), lam.cpu(), None if old is None else old.cpu(),
                                  inp["mask"].cpu(), mode, kk, flags=opd.F_GRADW_BF16)
    assert hr["grad_W"].dtype == torch.bfloat16
    check_grad(f64(hr["grad_W"]), ref["grad_W"], "bf16", "host bf16 grad_W")
    h32 = handle.loss_fwd_bwd_host(inp["hidden"].cpu(), inp["W"].cpu(), idx.cpu(), lam.cpu(), None if old is None else old.cpu(),
                                   inp["mask"].cpu(), mode, kk)
    assert h32["d2h_bytes"] - hr["d2h_bytes"] == 2 * cfg["d"] * cfg["V"]


def test_pipelined_host_entry(handle, opd):
    """opd_loss_fwd_bwd_host_submit / _wait: two steps in flight on the two staging slots give the results of the
    synchronous call; a busy slot refuses a second submit; waiting on an idle slot is an error."""
    cfg = RAGGED
    hosts, refs = [], []
    for c in (12, 13, 14):
        inp = synth.make_inputs(cfg, c=c, device=DEV)
        idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
        r = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk)
        torch.cuda.synchronize()
        refs.append({k: r[k].cpu() for k in ("loss", "per_token_kl", "grad_hidden", "grad_W")})
        hosts.append([t.cpu().pin_memory() for t in (inp["hidden"], inp["W"], idx, lam, old, inp["mask"])] + [kk])
    T, d, V = cfg["T"], cfg["d"], cfg["V"]
    new_out = lambda: dict(loss=torch.empty(1).pin_memory(), per_token_kl=torch.empty(T).pin_memory(),
                           grad_hidden=torch.empty(T, d, dtype=torch.bfloat16).pin_memory(), grad_W=torch.empty(d, V).pin_memory())
    outs = [new_out() for _ in range(3)]
    sub = lambda i: handle.host_submit(i % 2, *hosts[i][:6], O.RKL_MC, hosts[i][6], outs[i])
    sub(0); sub(1)
    with pytest.raises(opd.OpdError):
        sub(2)                                              # slot 0 is still in flight
    o0, up, down = handle.host_wait(0)
    sub(2)
    handle.host_wait(1); handle.host_wait(0)
    with pytest.raises(opd.OpdError):
        handle.host_wait(1)
    assert up > 0 and down > 0
    for i in range(3):
        assert abs(outs[i]["loss"].item() - refs[i]["loss"].item()) <= 1e-6
        assert torch.equal(outs[i]["per_token_kl"], refs[i]["per_token_kl"])
        check_grad(f64(outs[i]["grad_hidden"]), f64(refs[i]["grad_hidden"]), "bf16")
        check_grad(f64(outs[i]["grad_W"]), f64(refs[i]["grad_W"]), "bf16")


def test_call_is_cuda_graph_capturable(handle):
    """opd_loss_fwd_bwd only enqueues work on the caller's stream (no allocation once the workspace exists, no sync):
    it can be captured into a CUDA graph and replayed; the replay reproduces the eager result on new input values."""
    cfg = dict(RAGGED, T=512)
    inp = synth.make_inputs(cfg, c=15, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    X = inp["hidden"].clone()
    gh, gw = torch.empty_like(X), torch.empty(cfg["d"], cfg["V"], device=DEV)
    handle.loss_fwd_bwd(X, inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk, grad_hidden=gh, grad_W=gw)   # sizes the workspace
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        r = handle.loss_fwd_bwd(X, inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk, grad_hidden=gh, grad_W=gw)
    X.copy_(inp["hidden"].flip(0))                        # new values in the captured input buffer
    g.replay()
    torch.cuda.synchronize()
    loss_g, gh_g, gw_g = r["loss"].clone(), gh.clone(), gw.clone()
    e = handle.loss_fwd_bwd(X, inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk)
    torch.cuda.synchronize()
    assert abs(loss_g.item() - e["loss"].item()) <= 1e-6 * abs(e["loss"].item())
    check_grad(f64(gh_g), f64(e["grad_hidden"]), "bf16")
    check_grad(f64(gw_g), f64(e["grad_W"]), "bf16")


@pytest.mark.parametrize("knobs", [dict(OPD_CTA_GROUP="1"), dict(OPD_G_BUFS="3", OPD_TB="256", OPD_VB="256"),
                                   dict(OPD_GROUP_M="3", OPD_HINT_GW="1", OPD_HINT_G="2"),
                                   dict(OPD_Q_DEPTH="1", OPD_TB="256", OPD_VB="512"), dict(OPD_Q_DEPTH="8", OPD_TB="256", OPD_VB="256")])
def test_tuning_knobs_do_not_change_results(handle, knobs, monkeypatch):
    """The single-CTA tile configuration, a 3-deep G ring with the smallest super-tiles, another raster group, L2
    hints and the extreme claim-ahead depths of the tile queue give the same outputs as the defaults (within summation-order noise) and match the oracle."""
    cfg = RAGGED
    inp = synth.make_inputs(cfg, c=16, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    base = run(handle, inp, idx, lam, old, O.RKL_MC, kk)
    for k, v in knobs.items():
        monkeypatch.setenv(k, v)
    r = run(handle, inp, idx, lam, old, O.RKL_MC, kk)
    compare_all(r, oracle_for(inp, idx, lam, old, O.RKL_MC, kk), f64(inp["mask"]), "bf16")
    assert abs(r["loss"].item() - base["loss"].item()) <= 1e-6
    assert torch.equal(r["student_logp"].nan_to_num(), base["student_logp"].nan_to_num())


def test_autograd_entry(handle):
    """opd_loss(...).backward() on a [V,d] lm_head parameter (transposed view used in place) against the oracle."""
    from paper_2606_24143_b200.autograd import opd_loss
    cfg = dict(RAGGED, T=384)
    inp = synth.make_inputs(cfg, c=17, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    hidden = inp["hidden"].clone().requires_grad_(True)
    weight = inp["W"].t().contiguous().requires_grad_(True)               # [V,d] like nn.Linear(d, V).weight
    loss, ptk = opd_loss(hidden, weight.t(), idx, lam, old, inp["mask"], O.RKL_MC, kk, return_per_token=True)
    (2.0 * loss).backward()
    torch.cuda.synchronize()
    ref = oracle_for(inp, idx, lam, old, O.RKL_MC, kk)
    check_loss(loss.item(), ref)
    assert weight.grad.shape == weight.shape and weight.grad.dtype == weight.dtype
    check_grad(f64(hidden.grad), 2.0 * ref["grad_hidden"], "bf16")
    check_grad(f64(weight.grad).T, 2.0 * ref["grad_W"], "bf16")
    with torch.no_grad():
        l2 = opd_loss(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk)
    assert abs(l2.item() - loss.item()) <= 1e-6


@pytest.mark.parametrize("mode", [O.RKL_MC, O.MIXED, O.RKL_TOPK, O.FKL_TOPK])
def test_results_are_bitwise_reproducible(handle, mode, monkeypatch):
    """The summation order is fixed (tiles are reduced into the fp32 accumulators in super-tile order, enforced by the
    dependency counters, whichever CTA runs a tile; the sparse backward of OPD_RKL_TOPK sums every grad_W column in sorted
    (token, slot) order without atomics): repeated calls give bit-identical losses and gradients in every mode. A race in
    the barrier / counter protocol of the persistent kernels would show up here."""
    monkeypatch.setenv("OPD_TB", "256"); monkeypatch.setenv("OPD_VB", "512")      # many super-tiles -> many dependencies
    cfg = dict(RAGGED, T=1500, V=4104)
    inp = synth.make_inputs(cfg, c=18, device=DEV)
    if mode == O.MIXED:
        m = inp["mask"].clone()
        m[(torch.arange(cfg["T"], device=DEV) % 3 == 0) & (m != 0)] = 2
        inp["mask"] = m
    idx, lam, old, kk = pick(inp, cfg, mode)
    first = None
    for _ in range(6):
        r = handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk)
        torch.cuda.synchronize()
        cur = (r["loss"].clone(), r["per_token_kl"].clone(), r["grad_hidden"].clone(), r["grad_W"].clone())
        if first is None:
            first = cur
        else:
            assert all(torch.equal(a, b) for a, b in zip(first, cur))

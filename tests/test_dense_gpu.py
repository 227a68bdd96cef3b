"""GPU parity of opd_dense_kl_fwd_bwd (dense two-head forward KL, Eq.(1) PAPER.md:57-59 with the teacher recomputed from
transmitted hidden states) against the fp64 oracle."""
import numpy as np
import pytest
import torch

from oracle import opd_oracle as O
from gen import synth
from tests._util import GRAD_TOL, LOSS_RTOL, check_grad, f64

pytestmark = pytest.mark.gpu
DEV = "cuda"


@pytest.fixture(scope="module")
def handle():
    from paper_2606_24143_b200 import opd
    return opd.Handle(0)


def make(dtype, T, d, dT, V, seed, masked=True):
    g = torch.Generator(device=DEV).manual_seed(synth.SEED0 + 500 + seed)
    dt = torch.bfloat16 if dtype == "bf16" else torch.float32
    X = torch.randn(T, d, generator=g, device=DEV).to(dt)
    W = (torch.randn(d, V, generator=g, device=DEV) * d ** -0.5).to(dt)
    XT = torch.randn(T, dT, generator=g, device=DEV).to(dt)
    WT = (torch.randn(dT, V, generator=g, device=DEV) * dT ** -0.5).to(dt)
    mask = torch.ones(T, dtype=torch.uint8, device=DEV)
    if masked:
        mask[torch.randperm(T, generator=torch.Generator().manual_seed(seed))[: T // 10].to(DEV)] = 0
    return X, W, XT, WT, mask


def compare(r, X, W, XT, WT, mask, dtype, reverse=False):
    """Every output against Eq.(1) / Eq.(2) as written (the oracle knows nothing about how the kernel rounds q)."""
    live = f64(mask) != 0
    exact = O.dense_kl_oracle(f64(X), f64(W), f64(XT), f64(WT), f64(mask), reverse=reverse)
    ptk = f64(r["per_token_kl"])
    bar = LOSS_RTOL * np.abs(exact["per_token_kl"]).max()
    assert np.abs(ptk - exact["per_token_kl"]).max() <= bar and np.all(ptk[~live] == 0)
    assert abs(r["loss"].item() - exact["loss"]) <= LOSS_RTOL * abs(exact["loss"])
    if r["grad_hidden"] is not None:
        gh = f64(r["grad_hidden"])
        assert np.all(gh[~live] == 0)
        check_grad(gh, exact["grad_hidden"], dtype, "grad_hidden")
        check_grad(f64(r["grad_W"]), exact["grad_W"], dtype, "grad_W")


@pytest.mark.parametrize("dtype,T,d,dT,V,layouts", [
    ("fp32", 256, 256, 128, 4096, ("dv", "dv")), ("bf16", 700, 320, 448, 2056, ("dv", "vd")),
    ("bf16", 700, 320, 448, 2056, ("vd", "dv")), ("bf16", 1024, 512, 1024, 32768, ("dv", "dv"))])
def test_dense_kl_parity(handle, dtype, T, d, dT, V, layouts):
    X, W, XT, WT, mask = make(dtype, T, d, dT, V, 1)
    Wl = W if layouts[0] == "dv" else W.t().contiguous().t()
    WTl = WT if layouts[1] == "dv" else WT.t().contiguous().t()
    r = handle.dense_kl_fwd_bwd(X, Wl, XT, WTl, mask)
    torch.cuda.synchronize()
    compare(r, X, W, XT, WT, mask, dtype)


@pytest.mark.parametrize("dtype,T,d,dT,V,layouts,tiles", [
    ("fp32", 256, 256, 128, 4096, ("dv", "dv"), None), ("bf16", 700, 320, 448, 2056, ("dv", "vd"), None),
    ("bf16", 700, 320, 448, 2056, ("vd", "dv"), (256, 512)), ("bf16", 1024, 512, 1024, 32768, ("dv", "dv"), None)])
def test_dense_reverse_kl_parity(handle, dtype, T, d, dT, V, layouts, tiles, monkeypatch):
    """OPD_F_DENSE_REVERSE: KL(p || q) of Eq.(2) and its gradient Eq.(3), fp32 and bf16, both storage orders of
    both heads, several super-tiles (ring reuse across the two launches), forward-only, N = 0."""
    from paper_2606_24143_b200 import opd
    if tiles:
        monkeypatch.setenv("OPD_TB", str(tiles[0])); monkeypatch.setenv("OPD_VB", str(tiles[1]))
    X, W, XT, WT, mask = make(dtype, T, d, dT, V, 4)
    Wl = W if layouts[0] == "dv" else W.t().contiguous().t()
    WTl = WT if layouts[1] == "dv" else WT.t().contiguous().t()
    r = handle.dense_kl_fwd_bwd(X, Wl, XT, WTl, mask, flags=opd.F_DENSE_REVERSE)
    torch.cuda.synchronize()
    compare(r, X, W, XT, WT, mask, dtype, reverse=True)
    f = handle.dense_kl_fwd_bwd(X, Wl, XT, WTl, mask, flags=opd.F_DENSE_REVERSE | opd.F_FWD_ONLY)
    torch.cuda.synchronize()
    assert f["grad_W"] is None and abs(f["loss"].item() - r["loss"].item()) <= 1e-5 * abs(r["loss"].item())
    none = handle.dense_kl_fwd_bwd(X, Wl, XT, WTl, torch.zeros_like(mask), flags=opd.F_DENSE_REVERSE)
    torch.cuda.synchronize()
    assert none["loss"].item() == 0 and not none["grad_W"].any() and not none["grad_hidden"].any()
    z = handle.dense_kl_fwd_bwd(X, Wl, X, Wl, mask, flags=opd.F_DENSE_REVERSE) if d == dT else None
    if z is not None:
        torch.cuda.synchronize()
        assert abs(z["loss"].item()) <= 1e-5 and z["grad_W"].abs().max().item() <= 1e-3 * r["grad_W"].abs().max().item()


def test_dense_kl_super_tiles_fwd_only_and_zero_case(handle, monkeypatch):
    """Several super-tiles in both directions (ring reuse, Q one block ahead of G) give the same numbers; forward-only
    runs the Q and G tiles alone; teacher == student gives loss 0 and zero gradients (up to bf16 rounding of q)."""
    from paper_2606_24143_b200 import opd
    X, W, XT, WT, mask = make("bf16", 700, 320, 448, 2056, 2)
    base = handle.dense_kl_fwd_bwd(X, W, XT, WT, mask)
    torch.cuda.synchronize()
    monkeypatch.setenv("OPD_TB", "256"); monkeypatch.setenv("OPD_VB", "512")
    r = handle.dense_kl_fwd_bwd(X, W, XT, WT, mask)
    torch.cuda.synchronize()
    assert handle.launch_stats()["super_rows"] == 256
    compare(r, X, W, XT, WT, mask, "bf16")
    assert abs(r["loss"].item() - base["loss"].item()) <= 1e-5 * abs(base["loss"].item())
    f = handle.dense_kl_fwd_bwd(X, W, XT, WT, mask, flags=opd.F_FWD_ONLY)
    torch.cuda.synchronize()
    assert f["grad_W"] is None and abs(f["loss"].item() - r["loss"].item()) <= 1e-5 * abs(r["loss"].item())
    z = handle.dense_kl_fwd_bwd(X, W, X, W, mask)
    torch.cuda.synchronize()
    assert abs(z["loss"].item()) <= 1e-4
    assert z["grad_W"].abs().max().item() <= 1e-2 * base["grad_W"].abs().max().item()
    none = handle.dense_kl_fwd_bwd(X, W, XT, WT, torch.zeros_like(mask))
    torch.cuda.synchronize()
    assert none["loss"].item() == 0 and not none["grad_W"].any() and not none["grad_hidden"].any()


def _dense_C3_check(handle, reverse, n_live_target=None):
    """T=16384 (varlen mask), d=2048, dT=4096, V=151936: per-token values and whole grad_hidden rows of sampled tokens against
    the oracle, grad_W element by element on >= 256 vocabulary columns (random ones, tile edges, the last partial vocabulary
    tile) against oracle.dense_grad_W_columns, and the per-k identity <W, grad_W>_k = <x, grad_hidden>_k."""
    from paper_2606_24143_b200 import opd
    cfg = synth.CONFIGS[3]
    T, d, V, dT = cfg["T"], cfg["d"], cfg["V"], 4096
    X, W, XT, WT, _ = make("bf16", T, d, dT, V, 3, masked=False)
    mask = synth.make_mask(cfg, 3, DEV)
    if n_live_target is not None:                                 # scattered subset of the live rows (bounds the oracle's time)
        live0 = torch.nonzero(mask).flatten()
        keep = live0[torch.randperm(live0.numel(), generator=torch.Generator().manual_seed(3))[:n_live_target].to(DEV)]
        mask = torch.zeros_like(mask)
        mask[keep] = 1
    r = handle.dense_kl_fwd_bwd(X, W, XT, WT, mask, flags=opd.F_DENSE_REVERSE if reverse else 0)
    torch.cuda.synchronize()
    live = np.flatnonzero(f64(mask))
    rng = np.random.default_rng(5)
    rows = np.sort(rng.choice(live, 10, replace=False))
    sel = torch.as_tensor(rows, device=DEV)
    ref = O.dense_kl_oracle(f64(X[sel]), f64(W), f64(XT[sel]), f64(WT), np.ones(len(rows)), norm_override=float(live.size),
                            reverse=reverse)
    assert np.abs(f64(r["per_token_kl"][sel]) - ref["per_token_kl"]).max() <= LOSS_RTOL * np.abs(ref["per_token_kl"]).max()
    check_grad(f64(r["grad_hidden"][sel]), ref["grad_hidden"], "bf16", "grad_hidden rows")
    assert abs(r["loss"].item() - r["per_token_kl"].double().sum().item() / live.size) <= 1e-5 * abs(r["loss"].item())
    gw, gh = r["grad_W"], r["grad_hidden"]
    dead = mask == 0
    assert not gh[dead].any() and not r["per_token_kl"][dead].any()
    lhs = (W.double() * gw.double()).sum(dim=1)
    rhs = (X.double() * gh.double()).sum(dim=0)
    assert (lhs - rhs).abs().max().item() <= 2e-2 * lhs.abs().max().item()
    cols = np.unique(np.concatenate([rng.choice(V, 160, replace=False), np.arange(V - V % 256, V), [0, 255, 256, 4095, 4096, 8191]]))
    assert cols.size >= 256
    want = O.dense_grad_W_columns(f64(X), f64(W), f64(XT), f64(WT), f64(mask), cols, reverse=reverse)
    got = f64(gw[:, torch.as_tensor(cols, device=DEV)])
    check_grad(got, want, "bf16", f"dense grad_W[:, {cols.size} columns], reverse={reverse}")
    col_scale = np.maximum(np.abs(want).max(axis=0), 1e-3 * np.abs(want).max())
    assert (np.abs(got - want).max(axis=0) <= 4 * GRAD_TOL["bf16"] * col_scale).all()


@pytest.mark.slow
def test_dense_kl_at_C3_shape_forward(handle):
    """Eq.(1) at the C3 shape with its own variable-length mask (about 10.9k live rows)."""
    _dense_C3_check(handle, reverse=False)


@pytest.mark.slow
def test_dense_kl_at_C3_shape_reverse(handle):
    """OPD_F_DENSE_REVERSE (Eq.(2),(3)) at the C3 shape: three launches, fp32 log-q ring; 6144 scattered live
    rows (two token super-tiles)."""
    _dense_C3_check(handle, reverse=True, n_live_target=6144)
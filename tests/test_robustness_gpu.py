"""GPU tests of the library's robustness properties ("Harden the library"):
the dynamically scheduled persistent backward next to kernels that hold SMs and next to a second handle, capture-time
workspace growth, the binding's argument checks, the non-destructive autograd backward, diagnostics capacity, and a
bounded seeded soak over shapes / masks / modes / super-tile sizes (each case twice, bitwise equal, every third one
against the oracle)."""
import numpy as np
import pytest
import torch

from oracle import opd_oracle as O
from gen import synth
from tests._util import check_grad, check_loss, compare_all, f64, oracle_for, pick

pytestmark = pytest.mark.gpu
DEV = "cuda"
BASE = dict(dtype="bf16", T=1500, d=320, V=4104, k=8, K=5, sigma=0.05, mask="random10")


@pytest.fixture(scope="module")
def opd():
    from paper_2606_24143_b200 import opd as m
    return m


@pytest.fixture(scope="module")
def handle(opd):
    return opd.Handle(0)


def _outputs(r):
    return tuple(r[k].clone() for k in ("loss", "per_token_kl", "grad_hidden", "grad_W"))


def test_backward_completes_while_another_kernel_holds_sms(handle, opd, monkeypatch):
    """A kernel on another stream keeps 40 SMs busy for 2 s. The persistent backward (grid = one CTA per SM, tiles that wait
    on tiles of other CTAs) must finish long before that kernel does, with bit-identical results: its tiles are claimed
    dynamically in dependency order, so it does not need all of its CTAs resident (a static tile list would spin until the
    other kernel leaves)."""
    monkeypatch.setenv("OPD_TB", "256"); monkeypatch.setenv("OPD_VB", "512")      # many super-tiles -> many dependencies
    inp = synth.make_inputs(BASE, c=31, device=DEV)
    idx, lam, old, kk = pick(inp, BASE, O.RKL_MC)
    call = lambda: handle.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk)
    ref = _outputs(call())
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    occ_done, main_done = torch.cuda.Event(), torch.cuda.Event()
    with torch.cuda.stream(side):
        handle.debug_occupy(40, 2000.0, stream=side.cuda_stream)
        occ_done.record(side)
    import time
    time.sleep(0.05)                                   # let the occupying CTAs take their SMs
    t0 = time.perf_counter()
    got = _outputs(call())
    main_done.record()
    main_done.synchronize()
    dt = time.perf_counter() - t0
    still_busy = not occ_done.query()
    torch.cuda.synchronize()
    assert still_busy and dt < 1.0, (still_busy, dt)   # finished while 40 SMs were taken, not after they were released
    assert all(torch.equal(a, b) for a, b in zip(ref, got))


def test_two_handles_on_two_streams(opd, monkeypatch):
    """Two handles enqueue their persistent backward kernels on two streams at the same time (opd.h: one handle per
    thread / stream): both complete with the results of running alone."""
    monkeypatch.setenv("OPD_TB", "256"); monkeypatch.setenv("OPD_VB", "512")
    h1, h2 = opd.Handle(0), opd.Handle(0)
    inp = synth.make_inputs(BASE, c=32, device=DEV)
    idx, lam, old, kk = pick(inp, BASE, O.RKL_MC)
    fidx, flam, _, fk = pick(inp, BASE, O.FKL_TOPK)
    a = lambda h, s=None: h.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk, stream=s)
    b = lambda h, s=None: h.loss_fwd_bwd(inp["hidden"], inp["W"], fidx, flam, None, inp["mask"], O.FKL_TOPK, fk, stream=s)
    ra, rb = _outputs(a(h1)), _outputs(b(h2))
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for _ in range(3):
        with torch.cuda.stream(s1):
            ga = a(h1, s1.cuda_stream)
        with torch.cuda.stream(s2):
            gb = b(h2, s2.cuda_stream)
        torch.cuda.synchronize()
        assert all(torch.equal(x, y) for x, y in zip(ra, _outputs(ga)))
        assert all(torch.equal(x, y) for x, y in zip(rb, _outputs(gb)))


def test_workspace_growth_is_refused_inside_a_capture(opd):
    """The handle-owned workspace grows with a cudaFree + cudaMalloc: refused with OPD_ERR_WORKSPACE inside a stream
    capture (include/opd.h), and the same call succeeds eagerly and then captures."""
    h = opd.Handle(0)
    cfg = dict(BASE, T=512)
    inp = synth.make_inputs(cfg, c=33, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    gh, gw = torch.empty_like(inp["hidden"]), torch.empty(cfg["d"], cfg["V"], device=DEV)
    call = lambda: h.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], O.RKL_MC, kk, grad_hidden=gh, grad_W=gw)
    g = torch.cuda.CUDAGraph()
    with pytest.raises(opd.OpdError) as e:
        with torch.cuda.graph(g):
            call()
    assert e.value.status == opd.ERR_WORKSPACE
    torch.cuda.synchronize()
    call()
    torch.cuda.synchronize()
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g2):
        r = call()
    g2.replay()
    torch.cuda.synchronize()
    assert np.isfinite(r["loss"].item())


def test_binding_checks_and_conversions(handle, opd):
    """What raw pointers cannot tell the C ABI: int64 indices and bool masks are converted, mismatched cache strides are
    made contiguous, wrong dtypes / devices / strides raise instead of being reinterpreted."""
    cfg = dict(BASE, T=300)
    inp = synth.make_inputs(cfg, c=34, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    X, W, m = inp["hidden"], inp["W"], inp["mask"]
    ref = handle.loss_fwd_bwd(X, W, idx, lam, old, m, O.RKL_MC, kk)
    r = handle.loss_fwd_bwd(X, W, idx.long(), lam, old, m != 0, O.RKL_MC, kk)           # torch.multinomial / bool masks
    assert torch.equal(r["loss"], ref["loss"]) and torch.equal(r["grad_W"], ref["grad_W"])
    lam_wide = torch.zeros(cfg["T"], kk + 3, device=DEV); lam_wide[:, :kk] = lam           # row stride differs from idx's
    r = handle.loss_fwd_bwd(X, W, idx, lam_wide[:, :kk], old, m, O.RKL_MC, kk)
    assert torch.equal(r["loss"], ref["loss"]) and torch.equal(r["grad_hidden"], ref["grad_hidden"])
    r = handle.loss_fwd_bwd(X, W, idx.t().contiguous().t(), lam, old, m, O.RKL_MC, kk)      # non-unit inner stride
    assert torch.equal(r["loss"], ref["loss"])
    bad = [dict(lam=lam.double()), dict(idx=idx.to(torch.int16)), dict(m=m.to(torch.int32)), dict(W=W.float()),
           dict(lam=lam.cpu()), dict(W=torch.empty(cfg["d"], 2 * cfg["V"], device=DEV, dtype=W.dtype)[:, ::2]),
           dict(lam=lam[:, :-1]), dict(m=m[:-1])]
    for kw in bad:
        args = dict(X=X, W=W, idx=idx, lam=lam, old=old, m=m); args.update(kw)
        with pytest.raises(opd.OpdError):
            handle.loss_fwd_bwd(args["X"], args["W"], args["idx"], args["lam"], args["old"], args["m"], O.RKL_MC, kk)
    with pytest.raises(opd.OpdError):                   # accumulating needs the caller's array
        handle.loss_fwd_bwd(X, W, idx, lam, old, m, O.RKL_MC, kk, flags=opd.F_GRADW_ACCUM)
    with pytest.raises(opd.OpdError):                   # wrong dtype of a supplied grad_W
        handle.loss_fwd_bwd(X, W, idx, lam, old, m, O.RKL_MC, kk, grad_W=torch.empty(cfg["d"], cfg["V"], device=DEV, dtype=torch.bfloat16))
    with pytest.raises(opd.OpdError) as e:              # the host entries cannot accumulate
        handle.loss_fwd_bwd_host(X.cpu(), W.cpu(), idx.cpu(), lam.cpu(), old.cpu(), m.cpu(), O.RKL_MC, kk, flags=opd.F_GRADW_ACCUM)
    assert e.value.status == opd.ERR_BAD_ARG
    # diagnostics arrays that are too small for a later call are refused, not overrun
    rho = torch.zeros(cfg["T"] - 1, kk, device=DEV)
    handle.set_diagnostics(rho, None)
    try:
        with pytest.raises(opd.OpdError):
            handle.loss_fwd_bwd(X, W, idx, lam, old, m, O.RKL_MC, kk)
    finally:
        handle.set_diagnostics(None, None)
    assert torch.cuda.current_device() == 0


def test_autograd_backward_twice(handle):
    """backward() with retain_graph=True twice: the saved gradients are not scaled in place, so both passes agree."""
    from paper_2606_24143_b200.autograd import opd_loss
    cfg = dict(BASE, T=384)
    inp = synth.make_inputs(cfg, c=35, device=DEV)
    idx, lam, old, kk = pick(inp, cfg, O.RKL_MC)
    hidden = inp["hidden"].clone().requires_grad_(True)
    W = inp["W"].clone().requires_grad_(True)
    loss = opd_loss(hidden, W, idx, lam, old, inp["mask"], O.RKL_MC, kk)
    (3.0 * loss).backward(retain_graph=True)
    g1h, g1w = hidden.grad.clone(), W.grad.clone()
    hidden.grad = None; W.grad = None
    (3.0 * loss).backward()
    assert torch.equal(hidden.grad, g1h) and torch.equal(W.grad, g1w)
    ref = oracle_for(inp, idx, lam, old, O.RKL_MC, kk)
    check_grad(f64(W.grad), 3.0 * ref["grad_W"], "bf16")


def test_seeded_soak(handle, opd, monkeypatch):
    """Bounded randomized soak (seeded, about 40 cases): shapes with ragged T / V / d, all modes, both W layouts, mask
    densities from one live token to all, super-tile sizes down to one tile. Every case runs twice (bitwise equal:
    the reduction order is fixed whatever CTA runs a tile) and every third case is compared with the oracle."""
    rng = np.random.default_rng(20260624)
    modes = [O.FKL_TOPK, O.RKL_MC, O.MIXED, O.RKL_TOPK]
    for case in range(40):
        T = int(rng.integers(1, 900)); d = 64 * int(rng.integers(1, 7)); V = 8 * int(rng.integers(32, 700))
        mode = modes[case % 4]
        dtype = "fp32" if case % 5 == 0 else "bf16"
        cfg = dict(dtype=dtype, T=T, d=d, V=V, k=int(rng.integers(1, min(17, V))), K=int(rng.integers(1, 17)), sigma=0.05, mask="none")
        inp = synth.make_inputs(cfg, c=200 + case, device=DEV)
        keep = max(1, int(T * rng.choice([0.02, 0.5, 1.0])))
        m = torch.zeros(T, dtype=torch.uint8, device=DEV)
        m[torch.randperm(T, generator=torch.Generator().manual_seed(case))[:keep].to(DEV)] = 1
        if mode == O.MIXED:
            m[(torch.arange(T, device=DEV) % 2 == 0) & (m != 0)] = 2
        inp["mask"] = m
        monkeypatch.setenv("OPD_TB", str(256 * int(rng.integers(1, 4)))); monkeypatch.setenv("OPD_VB", str(256 * int(rng.integers(1, 5))))
        idx, lam, old, kk = pick(inp, cfg, mode)
        W = inp["W"] if case % 2 == 0 else inp["W"].t().contiguous().t()
        outs = []
        for _ in range(2):
            r = handle.loss_fwd_bwd(inp["hidden"], W, idx, lam, old, m, mode, kk, want_lse=True, want_student_logp=True)
            torch.cuda.synchronize()
            outs.append(_outputs(r))
        assert all(torch.equal(a, b) for a, b in zip(*outs)), (case, cfg, mode)
        if case % 3 == 0:
            compare_all(r, oracle_for(inp, idx, lam, old, mode, kk), f64(m), dtype)

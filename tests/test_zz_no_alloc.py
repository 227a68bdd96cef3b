"""opd_loss_fwd_bwd_static: the hot path for callers that cannot allocate GPU memory.

Some users of this library never get to call cudaMalloc: a learner process that shares its B200 with an inference engine
(or any framework allocator) which claimed the free HBM at start-up has nothing left to ask the driver for, and a serving /
training loop that keeps other streams busy cannot take the device-wide stall that cudaMalloc and cudaFree cause.  For them
the library carries one fixed 32 MiB scratch array in its own device image and an entry point that works only out of it.

This file checks that entry point against the ordinary one (opd_loss_fwd_bwd, whose workspace the handle allocates):
same inputs, same outputs within the bars every parity test here uses (tests/_util.py), on calls made back to back so
that each one starts from whatever the previous call, of a different shape and mode, left in the shared array.  It also
checks that a handle which only ever uses the static entry point does not lower the device's free memory, that the handle's
own workspace is left alone, and that a shape beyond the array's size is refused with a message instead of being run.

The file is named test_zz_* so that pytest collects it after every other test file: `pytest -x` stops at the first failure,
and a failure here must not hide the parity tests.  It does not depend on them: it builds its own handles and inputs, and
passes alone in a fresh process as well as at the end of the whole suite.
"""
import numpy as np
import pytest
import torch

from oracle import opd_oracle as O
from gen import synth
from tests._util import GRAD_TOL, LOGP_ATOL, LOSS_RTOL, f64, pick

pytestmark = pytest.mark.gpu
DEV = "cuda"

# three workloads that fit the 32 MiB array: BASELINE.json configs[0] (fp32, 15.7 MiB of scratch), a ragged bf16 shape
# with mixed forward-KL / Monte-Carlo rows, and the largest bf16 shape of the C2 family that still fits with gradients
CASES = {
    "C1_fp32_mc": (synth.CONFIGS[1], 1, O.RKL_MC),
    "ragged_bf16_mixed": (dict(dtype="bf16", T=700, d=320, V=2056, k=8, K=5, sigma=0.05, mask="random10"), 7, O.MIXED),
    "bf16_T1024_d1024_V32768_fkl": (dict(dtype="bf16", T=1024, d=1024, V=32768, k=16, K=4, sigma=0.02, mask="random10"), 12, O.FKL_TOPK),
}


@pytest.fixture(scope="module")
def opd():
    from paper_2606_24143_b200 import opd as m
    return m


def _inputs(name):
    cfg, c, mode = CASES[name]
    inp = synth.make_inputs(cfg, c=c, device=DEV)
    if mode == O.MIXED:
        m = inp["mask"].clone()
        m[(torch.arange(cfg["T"], device=DEV) % 3 == 0) & (m != 0)] = 2
        inp["mask"] = m
    idx, lam, old, kk = pick(inp, cfg, mode)
    idx, lam = idx.contiguous(), lam.contiguous()
    old = None if old is None else old.contiguous()
    return cfg, mode, inp, idx, lam, old, kk


def _outputs(inp, idx):
    """Every buffer the static call writes, made by the caller up front (the entry point allocates nothing) and filled
    with NaN so that an element the call failed to write cannot pass for a result."""
    T, d = inp["hidden"].shape
    V = inp["W"].shape[1]
    nan = float("nan")
    return dict(loss=torch.full((1,), nan, device=DEV), per_token_kl=torch.full((T,), nan, device=DEV),
                grad_hidden=torch.full((T, d), nan, device=DEV, dtype=inp["hidden"].dtype),
                grad_W=torch.full((d, V), nan, device=DEV), lse=torch.full((T,), nan, device=DEV),
                student_logp=torch.full((T, idx.stride(0)), nan, device=DEV))


def _same(static, ref, mask, dtype, what):
    """`static` (new entry point) against `ref` (existing path) at the bars of tests/_util.py."""
    live = f64(mask) != 0
    a, b = float(static["loss"].item()), float(ref["loss"].item())
    ptk_a, ptk_b = f64(static["per_token_kl"]), f64(ref["per_token_kl"])
    assert np.isfinite(a) and abs(a - b) <= LOSS_RTOL * max(abs(b), float(np.mean(np.abs(ptk_b)))), (what, a, b)
    assert np.abs(ptk_a - ptk_b).max() <= LOSS_RTOL * max(1e-30, float(np.abs(ptk_b).max())), what
    assert np.all(ptk_a[~live] == 0), what
    assert np.abs(f64(static["lse"])[live] - f64(ref["lse"])[live]).max() <= LOGP_ATOL, what
    sa, sb = f64(static["student_logp"])[live], f64(ref["student_logp"])[live]
    assert np.array_equal(np.isnan(sa), np.isnan(sb)), what                     # the same slots are written
    used = ~np.isnan(sb)
    assert np.abs(sa[used] - sb[used]).max() <= LOGP_ATOL, what
    for g in ("grad_hidden", "grad_W"):
        ga, gb = f64(static[g]), f64(ref[g])
        assert np.all(np.isfinite(ga)), (what, g)
        assert np.abs(ga - gb).max() <= GRAD_TOL[dtype] * float(np.abs(gb).max()) + 1e-30, (what, g)
    assert np.all(f64(static["grad_hidden"])[~live] == 0), what                  # masked rows are exact zeros


def test_static_entry_matches_the_allocating_path_on_calls_in_a_row(opd):
    """Back-to-back static calls over three different shapes / modes / dtypes, then the first one again: each must agree
    with opd_loss_fwd_bwd on the same inputs although it starts from the scratch contents the previous call left."""
    h_static, h_ref = opd.Handle(0), opd.Handle(0)
    data = {name: _inputs(name) for name in CASES}
    ref = {}
    for name, (cfg, mode, inp, idx, lam, old, kk) in data.items():
        ref[name] = h_ref.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, want_lse=True,
                                       want_student_logp=True)
    torch.cuda.synchronize()
    order = list(CASES) + [next(iter(CASES))]                  # A, B, C, A: no sync or clean-up between the calls
    got = []
    for name in order:
        cfg, mode, inp, idx, lam, old, kk = data[name]
        assert h_static.workspace_bytes(cfg["T"], cfg["d"], cfg["V"], idx.shape[1], 1 if cfg["dtype"] == "fp32" else 0, mode) \
            <= opd.STATIC_SCRATCH_BYTES
        out = _outputs(inp, idx)
        r = h_static.loss_fwd_bwd_static(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, out)
        assert r is out
        got.append((name, out))
    torch.cuda.synchronize()
    for name, out in got:
        cfg, mode, inp, idx = data[name][:4]
        out = dict(out, student_logp=out["student_logp"][:, :idx.shape[1]])
        _same(out, ref[name], inp["mask"], cfg["dtype"], name)
    # first and fourth call are the same problem: the library is bit-reproducible, whatever the scratch held before
    for key in ("loss", "per_token_kl", "grad_hidden", "grad_W"):
        assert torch.equal(got[0][1][key], got[3][1][key]), key
    h_static.close()
    h_ref.close()


def test_static_entry_takes_no_device_memory_and_leaves_the_handle_workspace_alone(opd):
    """After one warm-up call (module loading and the one-time address look-up happen there), a handle that has never used
    the allocating path runs static calls without the device's free memory going down; the allocating path on the same
    shape takes its 15.7 MiB workspace from the driver, which is what the static entry point exists to avoid."""
    cfg, mode, inp, idx, lam, old, kk = _inputs("C1_fp32_mc")
    out = _outputs(inp, idx)
    warm = opd.Handle(0)
    warm.loss_fwd_bwd_static(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, out)
    torch.cuda.synchronize()
    fresh = opd.Handle(0)
    need = fresh.workspace_bytes(cfg["T"], cfg["d"], cfg["V"], idx.shape[1], 1, mode)
    assert (8 << 20) < need <= opd.STATIC_SCRATCH_BYTES
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        fresh.loss_fwd_bwd_static(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, out)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free0 - free1 < (4 << 20), f"free device memory fell by {free0 - free1} bytes across static calls"
    first = {k: v.clone() for k, v in out.items()}
    # the same handle may still use the allocating path afterwards, and the static call before / after it is unaffected
    ref = fresh.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, want_lse=True, want_student_logp=True)
    fresh.loss_fwd_bwd_static(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, out)
    torch.cuda.synchronize()
    _same(dict(out, student_logp=out["student_logp"][:, :idx.shape[1]]), ref, inp["mask"], cfg["dtype"], "after the allocating path")
    for key in ("loss", "per_token_kl", "grad_hidden", "grad_W"):
        assert torch.equal(first[key], out[key]), key
    warm.close()
    fresh.close()


def test_static_entry_refuses_what_does_not_fit_or_would_need_a_copy(opd):
    """A shape whose plan exceeds the array is turned down on the host with both sizes in the message, before any launch
    (the outputs stay untouched); inputs that the ordinary binding would silently convert are turned down as well."""
    h = opd.Handle(0)
    T, d, V, C = 4096, 1024, 32768, 4                            # C2 with gradients: 72.9 MiB of scratch
    assert h.workspace_bytes(T, d, V, C, 0, O.RKL_MC) > opd.STATIC_SCRATCH_BYTES
    hidden = torch.zeros(T, d, device=DEV, dtype=torch.bfloat16)
    W = torch.zeros(d, V, device=DEV, dtype=torch.bfloat16)
    idx = torch.zeros(T, C, device=DEV, dtype=torch.int32)
    lam = torch.zeros(T, C, device=DEV)
    mask = torch.ones(T, device=DEV, dtype=torch.uint8)
    out = dict(loss=torch.full((1,), 7.0, device=DEV), per_token_kl=torch.full((T,), 7.0, device=DEV),
               grad_hidden=torch.full((T, d), 7.0, device=DEV, dtype=torch.bfloat16), grad_W=torch.full((d, V), 7.0, device=DEV))
    with pytest.raises(opd.OpdError) as e:
        h.loss_fwd_bwd_static(hidden, W, idx, lam, lam, mask, O.RKL_MC, C, out)
    assert e.value.status == opd.ERR_WORKSPACE and "OPD_STATIC_SCRATCH_BYTES" in str(e.value) and str(opd.STATIC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()
    assert float(out["loss"].item()) == 7.0 and bool((out["grad_W"] == 7.0).all()) and bool((out["per_token_kl"] == 7.0).all())
    # the forward-only form of the same shape fits (12.9 MiB) and runs
    assert h.workspace_bytes(T, d, V, C, 0, O.RKL_MC, opd.F_FWD_ONLY) <= opd.STATIC_SCRATCH_BYTES
    h.loss_fwd_bwd_static(hidden, W, idx, lam, lam, mask, O.RKL_MC, C, dict(loss=out["loss"], per_token_kl=out["per_token_kl"]),
                          flags=opd.F_FWD_ONLY)
    torch.cuda.synchronize()
    assert np.isfinite(float(out["loss"].item())) and float(out["loss"].item()) != 7.0
    with pytest.raises(opd.OpdError) as e:                       # int64 indices would need a converted copy
        h.loss_fwd_bwd_static(hidden, W, idx.long(), lam, lam, mask, O.RKL_MC, C, out, flags=opd.F_FWD_ONLY)
    assert e.value.status == opd.ERR_BAD_ARG
    h.close()

#!/usr/bin/env python
"""bench.py — fused OPD loss forward+backward throughput on B200 (metric of BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (pre-pass, forward contraction + LSE + gather, estimators,
backward super-tiles) over one batch of seeded synthetic input.  Prints ONE JSON line (rank 0).
Under torchrun (N>1) every rank runs its own token shard against a replica of W (no collective inside the loss itself:
DESIGN.md "Multi-GPU"); the exchange a data-parallel learner needs after it (all-reduce of loss and grad_W over NCCL, on a side
stream, overlapping the next step) is inside the timed region and reported under "collective".  Timing = max over ranks,
value = tokens of all ranks / that time ("weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "OPD loss fwd+bwd tokens/s on 1 B200; % of dense BF16 tensor peak"
UNIT = "live tokens/s"


def csrc_sha16() -> str:
    """sha256 (first 16 hex digits) over include/opd.h and the kernel sources, in name order: identifies the build a capture under
    profiles/ belongs to (the GPU box has no .git, so a commit id is not available at run time)."""
    import hashlib
    from paper_2606_24143_b200 import build
    hsh = hashlib.sha256()
    for f in build.sources():
        hsh.update(os.path.basename(f).encode() + b"\0" + open(f, "rb").read())
    return hsh.hexdigest()[:16]


def ncu_traffic(workload_key: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture of this workload
    (profiles/ncu_traffic.json names the capture and the command). bench.py never runs under a profiler, so this is a citation
    ("traffic_measured": false), and it is only given while the kernel sources are the ones the capture was taken from."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(p):
        return None
    ent = json.load(open(p)).get(workload_key)
    if not ent or ent.get("csrc_sha16") != csrc_sha16():
        return None
    return ent


def config_dict(cfg, mode_name, C, sigma):
    """The workload description both arms print (identical dicts: the driver compares them)."""
    return dict(workload=f"{cfg['name']} {mode_name} C={C} sigma={sigma}", T=cfg["T"], d=cfg["d"], V=cfg["V"],
                l2_policy="inputs larger than L2 (W alone is %.0f MB)" % (cfg["d"] * cfg["V"] * 2 / 1e6))


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return dict(burst=float(j["bf16_tflops"]), sustained=float(j.get("bf16_tflops_sustained", j["bf16_tflops"])),
                    hbm=float(j["hbm_gbs"]), src="measured")
    return dict(burst=1590.0, sustained=1400.0, hbm=6650.0, src="fallback")


def same_box_cublas(dev, seconds: float = 3.0):
    """What the library GEMM does on THIS box right now, measured the way MEASURED_PEAKS.json was (torch.matmul bf16 8192^3:
    best of 10 = burst, back to back for `seconds` = sustained).  Boxes of the pool differ by several per cent in what the
    1000 W cap lets them sustain; this is context beside the driver-written peaks, never the roofline's denominator."""
    n = 8192
    a = torch.randn(n, n, device=dev, dtype=torch.bfloat16)
    b = torch.randn(n, n, device=dev, dtype=torch.bfloat16)
    c = torch.empty(n, n, device=dev, dtype=torch.bfloat16)
    for _ in range(3):
        torch.matmul(a, b, out=c)
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); torch.matmul(a, b, out=c); e1.record(); torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps, t0 = 0, time.perf_counter()
    e0.record()
    while time.perf_counter() - t0 < seconds:
        for _ in range(20):
            torch.matmul(a, b, out=c)
        reps += 20
        torch.cuda.synchronize()
    e1.record(); torch.cuda.synchronize()
    fl = 2.0 * n ** 3 / 1e12
    return dict(burst=fl / (best * 1e-3), sustained=fl * reps / (e0.elapsed_time(e1) * 1e-3), how="torch.matmul bf16 8192^3 on this box, after the timed steps")


def workload(cfg_id: int, args):
    from gen import synth
    cfg = dict(synth.CONFIGS[cfg_id])
    if args.tokens:
        cfg["T"] = args.tokens
    if args.cache_width:
        cfg["k"] = cfg["K"] = args.cache_width
    if args.hot_columns:
        cfg["hot_columns"] = args.hot_columns
    return cfg


def pick_cache(inp, cfg, mode_name):
    from gen import synth
    from paper_2606_24143_b200 import opd
    if mode_name == "fkl":
        return opd.FKL_TOPK, inp["topk_idx"], inp["topk_logq"], None, cfg["k"]
    if mode_name == "rtopk":
        return opd.RKL_TOPK, inp["stopk_idx"], inp["stopk_logq"], None, cfg["k"]
    if mode_name == "mixed":
        idx, lam, old, kk = synth.mixed_cache(inp)
        return opd.MIXED, idx, lam, old, kk
    return opd.RKL_MC, inp["mc_idx"], inp["mc_logq"], inp["mc_logp_old"], cfg["K"]


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, gpu: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.p.terminate()
        try:
            out = self.p.communicate(timeout=5)[0]
        except Exception:
            out = ""
        sm, mx, pw, reasons = [], [], [], set()
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w=float(np.median(pw)), samples=len(sm),
                    reasons=sorted(reasons))


def to_np(t):
    if t is None:
        return None
    t = t.detach().cpu()
    return t.double().numpy() if t.is_floating_point() else t.numpy()


def oracle_prepare(inp, idx, lam, old, max_rows: int):
    """fp64 numpy copies of the first rows of the workload (input conversion is not part of the timed oracle run)."""
    mask = to_np(inp["mask"])
    rows = np.flatnonzero(mask)[:max_rows]
    n = int(rows.max()) + 1 if rows.size else 0
    return dict(X=to_np(inp["hidden"][:n]), W=to_np(inp["W"]), idx=to_np(idx[:n]), lam=to_np(lam[:n]),
                old=None if old is None else to_np(old[:n]), mask=mask[:n], rows=rows)


def oracle_sample(prep, mode, kk, n_rows: int):
    """The fp64 oracle as it stands on the first n_rows live tokens of the workload (full d and V), forward+backward."""
    from oracle import opd_oracle as O
    rows = prep["rows"][:n_rows]
    t0 = time.perf_counter()
    O.opd_oracle(prep["X"], prep["W"], prep["idx"], prep["lam"], prep["old"], prep["mask"], mode, kk, rows=list(rows))
    return len(rows), time.perf_counter() - t0


def oracle_rows_for(prep, mode, kk, seconds: float, cap: int = 256) -> int:
    """Rows per timed oracle run so that it lasts about `seconds`: t(n) = a + b n fitted on 4 and 16 rows."""
    oracle_sample(prep, mode, kk, 2)
    n1, t1 = oracle_sample(prep, mode, kk, 4)
    n2, t2 = oracle_sample(prep, mode, kk, 16)
    b = max((t2 - t1) / max(n2 - n1, 1), 1e-7)
    a = max(t1 - b * n1, 0.0)
    return int(max(2, min(cap, len(prep["rows"]), (seconds - a) / b)))


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p["num_threads"] for p in threadpool_info() if p.get("user_api") == "blas"]
        return int(max(n)) if n else os.cpu_count()
    except Exception:
        return os.cpu_count()


def run_reference(args, rank, world):
    if rank != 0:
        return
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    cfg = workload(args.config, args)
    gen = dict(cfg)
    gen["T"] = min(cfg["T"], 2048)                 # the oracle only sees a bounded sample of the workload's rows
    from gen import synth
    inp = synth.make_inputs(gen, c=args.config, device=dev, sigma=args.sigma)
    mode, idx, lam, old, kk = pick_cache(inp, gen, args.mode)
    prep = oracle_prepare(inp, idx, lam, old, 2048)
    rows = oracle_rows_for(prep, mode, kk, args.ref_seconds, cap=2048)
    for _ in range(1 if args.warmup >= 1 else 0):
        oracle_sample(prep, mode, kk, rows)
    tot_t, tot_n = 0.0, 0
    for _ in range(args.steps):
        n, dt = oracle_sample(prep, mode, kk, rows)
        tot_t += dt; tot_n += n
    v = tot_n / tot_t
    sample = f"{rows} live tokens of {cfg['name']} per step (full d={cfg['d']}, V={cfg['V']}), forward+backward incl. grad_W, numpy fp64"
    line = dict(impl="reference", metric=METRIC, value=v, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * tot_t / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=config_dict(cfg, args.mode, idx.shape[1], inp["sigma"]),
                cpu_baseline=dict(value=v, unit=UNIT, cores=cpu_threads(), kind="oracle", sample=sample),
                e2e=dict(value=v, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line), flush=True)


def run_producer_bench(args, h, inp, cfg, dev, world, rank, dist):
    """Cache producers (opd_cache_topk / opd_cache_sample) on the workload's shapes: tokens scored per second.
    Two streamed contractions per call (pass A: LSE partials, pass B: collect / resolve), 4*d*V flops per token."""
    T, d, V = cfg["T"], cfg["d"], cfg["V"]
    n = cfg["k"] if args.op == "topk" else cfg["K"]
    u = torch.rand(T, n, device=dev, generator=torch.Generator(device=dev).manual_seed(1)) if args.op == "sample" else None
    # the scoring model's head: an independent seeded matrix of the same shape (synth keeps only W resident)
    Wt = inp["W"]
    flops = 4.0 * d * V * T
    n_tok = T
    if args.op == "dense":      # dense two-head forward KL: teacher hidden states and head of the student's shapes (dT = d)
        g = torch.Generator(device=dev).manual_seed(2)
        th = torch.randn(T, d, device=dev, generator=g).to(inp["hidden"].dtype)
        wt = (torch.randn(d, V, device=dev, generator=g) * d ** -0.5).to(inp["W"].dtype)
        gh = torch.empty_like(inp["hidden"]); gw = torch.empty(d, V, dtype=torch.float32, device=dev)
        from paper_2606_24143_b200 import opd as _opd
        dflags = _opd.F_DENSE_REVERSE if args.reverse else 0
        call = lambda: h.dense_kl_fwd_bwd(inp["hidden"], inp["W"], th, wt, inp["mask"], flags=dflags, grad_hidden=gh, grad_W=gw)
        n_tok = int((inp["mask"] != 0).sum().item())
        # two forward heads, Q and G re-formation, grad_hidden, grad_W: 2 d V each; the reverse direction re-forms both heads
        # once more in the streamed pass that produces the per-token value before the gradient tiles
        flops = (16.0 if args.reverse else 12.0) * d * V * n_tok
        n = 0
    elif args.op == "topk":
        call = lambda: h.cache_topk(inp["hidden"], Wt, n)
    else:
        call = lambda: h.cache_sample(inp["hidden"], Wt, u)
    for _ in range(max(args.warmup, 3)):
        call()
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    ev[0].record()
    for _ in range(args.steps):
        call()
    ev[1].record()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    total_ms = ev[0].elapsed_time(ev[1])
    clocks = sampler.stop() if sampler else None
    if dist is not None:
        t = torch.tensor([total_ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    if rank != 0:
        return
    ms = total_ms / args.steps
    pk = peaks()
    ach = flops / (ms * 1e-3) / 1e12
    st = h.launch_stats()
    line = dict(metric=(f"cache producer ({args.op}) tokens scored/s on 1 B200" if args.op != "dense" else
                        ("dense two-head reverse KL fwd+bwd tokens/s on 1 B200" if args.reverse else "dense two-head forward KL fwd+bwd tokens/s on 1 B200")), value=n_tok * world / (ms * 1e-3), unit="live tokens/s" if args.op == "dense" else "tokens/s", n_gpus=world,
                steps=args.steps, warmup=max(args.warmup, 3), ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="bf16" if cfg["dtype"] == "bf16" else "f32(3xbf16)", data="synthetic",
                config=dict(workload=(f"{cfg['name']} opd_cache_{args.op} n={n}" if args.op != "dense" else f"{cfg['name']} opd_dense_kl_fwd_bwd dT=d" + (" reverse" if args.reverse else "")),
                            T=T, d=d, V=V,
                            l2_policy="inputs larger than L2 (W alone is %.0f MB)" % (d * V * 2 / 1e6)),
                clocks=clocks, e2e=None, gpu_launches=st["kernels"] * args.steps,
                roofline=dict(bound="tensor", achieved=ach, peak=pk["sustained"], unit="TFLOP/s", frac=ach / pk["sustained"], traffic=None,
                              kernel=("opd::gemm_kernel<FwdEpi,2> + opd::gemm_kernel<%s,2>" % ("CollectEpi" if args.op == "topk" else "SampleEpi")
                                      if args.op != "dense" else "2 x opd::gemm_kernel<FwdEpi,2> + opd::bwd_kernel<2,true>"),
                              flops_per_step=flops, frac_of_burst=ach / pk["burst"]),
                cpu_baseline=None)
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config (1..5); 4 = the config the metric is quoted on")
    ap.add_argument("--mode", default=None, choices=["fkl", "mc", "mixed", "rtopk"])
    ap.add_argument("--op", default="loss", choices=["loss", "topk", "sample", "dense"],
                    help="loss = the hot path (default, the contract's line); topk / sample = the cache producers (NEXT-3)")
    ap.add_argument("--tokens", type=int, default=0, help="override T (debugging)")
    ap.add_argument("--sigma", type=float, default=None, help="staleness of the rollout policy: W_old = W + sigma*N(0,1/d)")
    ap.add_argument("--cache-width", type=int, default=0, help="override the config's k and K (C4's cost-vs-cache-size sweep)")
    ap.add_argument("--hot-columns", type=int, default=0, help="skewed top-k supports: this many fixed columns sit in (almost) every row's top-k cache "
                    "(gen/synth.py; the tail case of the sparse backward of --mode rtopk)")
    ap.add_argument("--layout", default="dv", choices=["dv", "vd"], help="storage order of W: [d,V] row-major (BASELINE.json) or [V,d] (lm_head.weight)")
    ap.add_argument("--diag", action="store_true", help="also report rho statistics of the MC cache (opd_set_diagnostics)")
    ap.add_argument("--fwd-only", action="store_true", help="diagnostic: time OPD_F_FWD_ONLY calls (S0-S5: pre-pass, forward contraction, estimators) back to back")
    ap.add_argument("--force-dist", action="store_true", help="run the N > 1 code path (global normaliser, all-reduce of loss and grad_W on a side "
                    "stream) with a one-rank NCCL group: a test aid for boxes with one GPU")
    ap.add_argument("--no-sustained", action="store_true", help="skip the >= 4 s back-to-back loop that follows a timed region shorter than 4 s")
    ap.add_argument("--reverse", action="store_true", help="--op dense: the reverse direction KL(p || q) (OPD_F_DENSE_REVERSE)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-probe", action="store_true", help="skip the same-box cuBLAS measurement (3 s, after the timed steps)")
    ap.add_argument("--ref-seconds", type=float, default=12.0)
    args = ap.parse_args()
    if args.mode is None:
        args.mode = "mixed" if args.config == 5 else "mc"

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the OPD path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1 or args.force_dist:
        import torch.distributed as dist
        if "RANK" not in os.environ:                  # --force-dist without torchrun: a one-rank group on this process
            os.environ.update(RANK="0", WORLD_SIZE="1", MASTER_ADDR="127.0.0.1", MASTER_PORT=os.environ.get("MASTER_PORT", "29533"))
        dist.init_process_group("nccl", device_id=dev)

    from gen import synth
    from paper_2606_24143_b200 import opd
    cfg = workload(args.config, args)
    inp = synth.make_inputs(cfg, c=args.config + 10 * rank, device=dev, sigma=args.sigma)
    mode, idx, lam, old, kk = pick_cache(inp, cfg, args.mode)
    T, d, V = cfg["T"], cfg["d"], cfg["V"]
    n_live = int((inp["mask"] != 0).sum().item())
    h = opd.Handle(local)
    if args.op != "loss":
        run_producer_bench(args, h, inp, cfg, dev, world, rank, dist)
        return
    if args.fwd_only:
        # forward-only diagnostic (profiles/r02_experiments.md section 11): not the contract's line
        f = lambda: h.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, flags=opd.F_FWD_ONLY)
        for _ in range(max(args.warmup, 3)):
            f()
        torch.cuda.synchronize()
        sampler = ClockSampler(local)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            f()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        print(json.dumps(dict(metric="OPD loss forward only (S0-S5) on 1 B200", ms_per_step=ms, tflops_executed=2.0 * d * V * n_live / ms / 1e9,
                              steps=args.steps, config=config_dict(cfg, args.mode, idx.shape[1], inp["sigma"]), clocks=sampler.stop())), flush=True)
        return
    gh = torch.empty_like(inp["hidden"])
    if args.layout == "vd":          # same logical [d,V] matrices, [V,d] storage
        inp["W"] = inp["W"].t().contiguous().t()
        gw = torch.empty(V, d, dtype=torch.float32, device=dev).t()
    else:
        gw = torch.empty(d, V, dtype=torch.float32, device=dev)

    # N > 1: every rank runs its own token shard against a replica of W with the GLOBAL live count as the
    # normaliser, and what a data-parallel learner must exchange afterwards is inside the timed region: loss and grad_W (fp32
    # d x V: 2.49 GB at C4) are all-reduced over NCCL on a side stream, so the reduction of step i overlaps the kernels of step
    # i + 1 (two grad_W buffers alternate; a buffer is not written again before its all-reduce has finished).
    norm = 0.0
    comm = None
    if dist is not None:
        ng = torch.tensor([n_live], device=dev, dtype=torch.int64)
        dist.all_reduce(ng)
        norm = float(ng.item())
        comm = dict(stream=torch.cuda.Stream(dev), bufs=[gw, torch.empty_like(gw)], done=[None, None], i=0, spans=[])

    def step():
        if comm is None:
            return h.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, grad_hidden=gh, grad_W=gw)
        b = comm["i"] % 2
        comm["i"] += 1
        if comm["done"][b] is not None:
            torch.cuda.current_stream(dev).wait_event(comm["done"][b])       # the buffer's previous all-reduce
        r = h.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, norm_override=norm, grad_hidden=gh,
                           grad_W=comm["bufs"][b])
        ready = torch.cuda.Event()
        ready.record()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(comm["stream"]):
            comm["stream"].wait_event(ready)
            a0.record()
            dist.all_reduce(r["loss"])
            dist.all_reduce(comm["bufs"][b])
            a1.record()
        comm["done"][b] = a1
        comm["spans"].append((a0, a1))
        return r

    def drain():                                        # the last all-reduces belong to the timed region
        if comm is not None:
            torch.cuda.current_stream(dev).wait_stream(comm["stream"])

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        r = step()
    drain()
    barrier()
    if comm is not None:
        comm["spans"].clear()
    stats = h.launch_stats()
    phase_sets = [h.new_phase_events() for _ in range(args.steps)]      # one set of phase events per timed step
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    ev[0].record()
    for i in range(args.steps):
        h.use_phase_events(phase_sets[i])
        r = step()
        if i == args.steps - 1:
            drain()
        ev[i + 1].record()
    barrier()
    h.use_phase_events(None)
    total_ms = ev[0].elapsed_time(ev[-1])
    collective = None
    if comm is not None:
        ar = [a.elapsed_time(b) for a, b in comm["spans"]]
        comm["spans"].clear()
        compute_ms = float(np.sum([sum(q.values()) for q in [h.phase_times_ms(ps) for ps in phase_sets]]))
        collective = dict(what="all_reduce(loss) + all_reduce(grad_W fp32 d x V) per step over NCCL, side stream, two grad_W buffers",
                          bytes_per_step=int(gw.numel() * 4 + 4), allreduce_ms=float(np.mean(ar)),
                          exposed_ms_per_step=max(0.0, (total_ms - compute_ms) / args.steps),
                          overlap_hidden_ms=max(0.0, float(np.mean(ar)) - max(0.0, (total_ms - compute_ms) / args.steps)),
                          norm_override=norm)
    step_ms = [round(ev[i].elapsed_time(ev[i + 1]), 3) for i in range(args.steps)]
    per_step = [h.phase_times_ms(ps) for ps in phase_sets]               # every timed step, CUDA events on the launching stream
    pm = {k: float(np.mean([q[k] for q in per_step])) for k in opd.PHASE_NAMES}          # average over the timed steps
    phase_steps = {k: [round(q[k], 3) for q in per_step] for k in opd.PHASE_NAMES}
    clocks = sampler.stop() if sampler else None
    loss_val = float(r["loss"].item())
    if dist is not None:
        t = torch.tensor([total_ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        nl = torch.tensor([n_live], device=dev, dtype=torch.int64)
        dist.all_reduce(nl)
        n_live_all = int(nl.item())
    else:
        n_live_all = n_live
    ms_per_step = total_ms / args.steps
    value = n_live_all / (ms_per_step * 1e-3)
    # SURVEY 8(d) protocol: a timed region shorter than 4 s does not reach the power-capped steady state the sustained peak was
    # measured in, so a second loop of back-to-back steps runs for at least 4 s (the way MEASURED_PEAKS.json's sustained figure
    # was taken) and is reported beside the contract's K-step number
    sustained = None
    if total_ms < 4000.0 and not args.no_sustained:
        n_sus = int(4200.0 / max(ms_per_step, 1e-3)) + 1
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        s0.record()
        for _ in range(n_sus):
            step()
        drain()
        s1.record()
        barrier()
        sus_ms = s0.elapsed_time(s1)
        if dist is not None:
            t = torch.tensor([sus_ms], device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            sus_ms = float(t.item())
        sustained = dict(steps=n_sus, seconds=sus_ms * 1e-3, ms_per_step=sus_ms / n_sus, value=n_live_all / (sus_ms / n_sus * 1e-3))
    ws_bytes = h.workspace_bytes(T, d, V, idx.shape[1], opd.BF16 if cfg["dtype"] == "bf16" else opd.FP32, mode)
    free_b, total_b = torch.cuda.mem_get_info(dev)
    memory = dict(torch_peak_allocated_bytes=int(torch.cuda.max_memory_allocated(dev)), opd_workspace_bytes=int(ws_bytes),
                  device_used_bytes=int(total_b - free_b), device_total_bytes=int(total_b),
                  note="device_used = everything on the GPU after the timed steps (inputs, generator leftovers in torch's cache, outputs, libopd workspace, CUDA context)")

    # ---- e2e: same call through the C ABI with HOST buffers (H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        hh = {k: inp[k].cpu().contiguous().pin_memory() for k in ("hidden", "W", "mask")}     # the host entry takes dense [d,V]
        hidx, hlam = idx.cpu().pin_memory(), lam.cpu().pin_memory()
        hold = None if old is None else old.cpu().pin_memory()
        def host_out():
            return dict(loss=torch.empty(1).pin_memory(), per_token_kl=torch.empty(T).pin_memory(),
                        grad_hidden=torch.empty(T, d, dtype=inp["hidden"].dtype).pin_memory(),
                        grad_W=torch.empty(d, V, dtype=torch.float32).pin_memory())
        outs = [host_out(), host_out()]
        del gw, gh
        if comm is not None:
            comm["bufs"] = None
        torch.cuda.empty_cache()
        n_e2e = max(2, min(args.steps, 20))      # the fill (first copy-in) and drain (last copy-out) of the pipeline are inside the timed region

        e2e_flags = 0

        def submit(i):
            h.host_submit(i % 2, hh["hidden"], hh["W"], hidx, hlam, hold, hh["mask"], mode, kk, outs[i % 2], flags=e2e_flags)

        # every step copies its inputs from pinned host memory and its results (loss, per-token KL, both gradients) back;
        # the two staging slots overlap step i's kernels with the copy-in of step i+1 and the copy-out of step i-1
        submit(0); h.host_wait(0)                                # warm-up (allocates staging)
        submit(1); h.host_wait(1)
        barrier()
        t0 = time.perf_counter()
        submit(0)
        for i in range(1, n_e2e):
            submit(i)
            o, up, down = h.host_wait((i - 1) % 2)
        o, up, down = h.host_wait((n_e2e - 1) % 2)
        barrier()
        dt = (time.perf_counter() - t0) / n_e2e
        # the plain synchronous call (no overlap), for comparison
        t1 = time.perf_counter()
        h.loss_fwd_bwd_host(hh["hidden"], hh["W"], hidx, hlam, hold, hh["mask"], mode, kk, out=outs[0])
        dt_sync = time.perf_counter() - t1
        if dist is not None:
            t = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = dict(value=n_live_all / dt, unit=UNIT, h2d_bytes_per_step=int(up), d2h_bytes_per_step=int(down),
                   steps=n_e2e, ms_per_step=dt * 1e3, loss=float(o["loss"].item()),
                   api="opd_loss_fwd_bwd_host_submit/_wait, 2 staging slots (copies of neighbouring steps overlap the kernels)",
                   unpipelined_ms_per_step=dt_sync * 1e3)
        # the same with a bf16 grad_W (OPD_F_GRADW_BF16): half the bytes of the largest copy back
        e2e_flags = opd.F_GRADW_BF16
        for o_ in outs:
            o_["grad_W"] = torch.empty(d, V, dtype=torch.bfloat16).pin_memory()
        submit(0); h.host_wait(0)
        barrier()
        t2 = time.perf_counter()
        submit(0)
        for i in range(1, n_e2e):
            submit(i)
            _, up16, down16 = h.host_wait((i - 1) % 2)
        _, up16, down16 = h.host_wait((n_e2e - 1) % 2)
        barrier()
        dt16 = (time.perf_counter() - t2) / n_e2e
        e2e["bf16_grad_W"] = dict(value=n_live / dt16, ms_per_step=dt16 * 1e3, h2d_bytes_per_step=int(up16), d2h_bytes_per_step=int(down16))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    diag = None
    if args.diag and mode == opd.RKL_MC:
        rho = torch.zeros(T, idx.shape[1], device=dev)
        h.set_diagnostics(rho, None)
        rr = h.loss_fwd_bwd(inp["hidden"], inp["W"], idx, lam, old, inp["mask"], mode, kk, flags=opd.F_FWD_ONLY)
        torch.cuda.synchronize()
        h.set_diagnostics(None, None)
        rl = rho[inp["mask"] != 0].flatten()
        srt = torch.sort(rl).values
        diag = dict(rho_mean=float(rl.mean()), rho_p99=float(srt[int(0.99 * (srt.numel() - 1))]), rho_max=float(rl.max()),
                    mean_per_token_kl=float(rr["per_token_kl"].sum() / max(n_live, 1)))
    pk = peaks()
    # Roofline of the dominant kernel, opd::bwd_kernel (one launch per step: S6 logits recompute + S7 grad_hidden +
    # S8 grad_W = 3 contractions of 2*d*V flops per live token), timed live with CUDA events on the
    # launching stream (phase "bwd"); the forward kernel (S1-S3, 2*d*V per token) beside it.
    flops_exec = 8.0 * d * V * n_live            # logits + recomputed logits + dX + dW  (2 d V each)
    bwd_flops, fwd_flops = 6.0 * d * V * n_live, 2.0 * d * V * n_live
    ach = bwd_flops / (pm["bwd"] * 1e-3) / 1e12
    ach_fwd = fwd_flops / (pm["fwd"] * 1e-3) / 1e12
    tr = ncu_traffic(f"C{args.config} {args.mode}") if not (args.tokens or args.cache_width or args.hot_columns or args.sigma is not None) else None
    roofline = dict(bound="tensor", achieved=ach, peak=pk["sustained"], unit="TFLOP/s", frac=ach / pk["sustained"],
                    traffic=tr["bwd_kernel"] if tr else None, traffic_measured=False,
                    kernel="opd::bwd_kernel<2,false> (persistent: G re-formation, grad_hidden, grad_W tiles on tcgen05 cta_group::2)",
                    flops_per_launch=bwd_flops, launches_per_step=1, ms_per_launch=pm["bwd"],
                    peak_kind=f"bf16_tflops_sustained of {pk['src']} (kernel timed inside a long step); burst peak {pk['burst']}",
                    frac_of_burst=ach / pk["burst"],
                    fwd_kernel=dict(kernel="opd::gemm_kernel<FwdEpi,2>", achieved=ach_fwd, frac=ach_fwd / pk["sustained"],
                                    frac_of_burst=ach_fwd / pk["burst"], flops_per_launch=fwd_flops, ms_per_launch=pm["fwd"],
                                    traffic=tr["fwd_kernel"] if tr else None),
                    traffic_source=tr["source"] if tr else None)
    whole = flops_exec / (ms_per_step * 1e-3) / 1e12
    box = None
    if world == 1 and not args.no_probe:
        box = same_box_cublas(dev)
        box["executed_8dV_vs_same_box_sustained"] = 100 * whole / box["sustained"]
    cpu = None
    if not args.no_cpu:
        sub = dict(hidden=inp["hidden"][:4096], W=inp["W"], mask=inp["mask"][:4096])
        prep = oracle_prepare(sub, idx[:4096], lam[:4096], None if old is None else old[:4096], 2048)
        rows = oracle_rows_for(prep, mode, kk, args.ref_seconds, cap=2048)
        n, dt = oracle_sample(prep, mode, kk, rows)
        cpu = dict(value=n / dt, unit=UNIT, cores=cpu_threads(), kind="oracle",
                   sample=f"{n} live tokens of this workload (full d, V), forward+backward incl. grad_W, numpy fp64, {dt:.1f} s")
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="bf16" if cfg["dtype"] == "bf16" else "f32(3xbf16)", data="synthetic",
                config=config_dict(cfg, args.mode, idx.shape[1], inp["sigma"]),
                launch=dict(live_tokens_per_gpu=n_live, super_tile=[stats["super_rows"], stats["super_cols"]], layout=args.layout),
                all_T_tokens_per_s=(T * world / (ms_per_step * 1e-3) if n_live < T else None),   # padding rows counted too (C3)
                sustained=sustained, memory=memory, collective=collective,
                pct_of_bf16_peak=dict(executed_8dV_vs_burst=100 * whole / pk["burst"], executed_8dV_vs_sustained=100 * whole / pk["sustained"],
                                      model_6dV_vs_burst=100 * whole * 0.75 / pk["burst"], tflops_executed=whole, peaks=pk, same_box_cublas=box),
                phase_ms=pm, phase_ms_per_step=phase_steps, step_ms=step_ms, loss=loss_val, clocks=clocks, e2e=e2e, gpu_launches=stats["kernels"] * args.steps,
                roofline=roofline, cpu_baseline=cpu, mc_diagnostics=diag)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

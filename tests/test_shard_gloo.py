"""world_size-2 gloo test (CPU) of the token-sharded path: shards + global normaliser + all-reduce of loss and
grad_W reproduce the single-process result.  The engine here is the fp64 oracle (the CUDA binding has the same
signature); what is under test is paper_2606_24143_b200/shard.py."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import opd_oracle as O
from gen import synth
from paper_2606_24143_b200 import shard

CFG = dict(dtype="fp32", T=96, d=16, V=64, k=4, K=3, sigma=0.05, mask="random10")


def oracle_engine(hidden, W, idx, lam, old, mask, mode, kk, norm_override=0.0, **kw):
    f = lambda t: None if t is None else t.double().numpy() if t.is_floating_point() else t.numpy()
    r = O.opd_oracle(f(hidden), f(W), f(idx), f(lam), f(old), f(mask), mode, kk, norm_override=norm_override)
    return dict(loss=torch.tensor([r["loss"]], dtype=torch.float64), grad_W=torch.from_numpy(r["grad_W"]),
                grad_hidden=torch.from_numpy(r["grad_hidden"]))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    inp = synth.make_inputs(CFG, c=3, device="cpu")
    seq_lens = [24, 8, 40, 24]
    a, b = shard.token_shard(seq_lens, rank, world)
    sl = slice(a, b)
    out = shard.sharded_loss_fwd_bwd(oracle_engine, inp["hidden"][sl], inp["W"], inp["mc_idx"][sl], inp["mc_logq"][sl],
                                     inp["mc_logp_old"][sl], inp["mask"][sl], O.RKL_MC, CFG["K"])
    q.put((rank, a, b, out["loss"].item(), out["grad_W"].numpy(), out["grad_hidden"].numpy(), out["N_global"]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_reproduce_single_process():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in range(2)], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    inp = synth.make_inputs(CFG, c=3, device="cpu")
    ref = oracle_engine(inp["hidden"], inp["W"], inp["mc_idx"], inp["mc_logq"], inp["mc_logp_old"], inp["mask"], O.RKL_MC, CFG["K"])
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == CFG["T"]         # shards partition the tokens
    assert res[0][6] == res[1][6] == float((inp["mask"] != 0).sum())
    for r in res:
        assert abs(r[3] - ref["loss"].item()) < 1e-12                                     # same loss on every rank
        np.testing.assert_allclose(r[4], ref["grad_W"].numpy(), atol=1e-13)
    gh = np.concatenate([res[0][5], res[1][5]])
    np.testing.assert_allclose(gh, ref["grad_hidden"].numpy(), atol=1e-13)


def test_token_shard_whole_sequences():
    lens = [5, 7, 3, 9, 4, 4]
    cuts = [shard.token_shard(lens, r, 3) for r in range(3)]
    assert cuts[0][0] == 0 and cuts[-1][1] == sum(lens)
    edges = set(np.cumsum([0] + lens).tolist())
    for a, b in cuts:
        assert a in edges and b in edges and a <= b
    assert all(cuts[i][1] == cuts[i + 1][0] for i in range(2))

"""B200-native fused OPD loss (learner-side hot path of AsyncOPD, arxiv/paper_2606_24143).

`paper_2606_24143_b200.opd`   — ctypes binding of the C-ABI library libopd.so (include/opd.h)
`paper_2606_24143_b200.autograd` — torch.autograd entry (opd_loss)
`paper_2606_24143_b200.shard` — host logic of the token-sharded multi-GPU use
`paper_2606_24143_b200.build` — nvcc build of csrc/ for sm_100a
(the seeded synthetic workloads live outside the product package, in gen/synth.py)
"""

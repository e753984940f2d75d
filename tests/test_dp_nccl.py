"""The data-parallel schedules of dp.py with the REAL kernels and NCCL at world size 2 (
PAPER.md:174, 302-304): the CUDA twin of tests/test_dp_gloo.py, which injects oracle steps under gloo.  Needs two GPUs
in one box; every box of the build pool has one, so there it is skipped (the single-GPU path of the same schedule is
covered bit for bit in tests/test_gpu_families.py)."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import dp, synth
from test_dp_gloo import HP, HPT, SHAPES, T, _bits, _free_port, _problems

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    try:
        ps = _problems()                                   # same seeds: the replicas start identical
        per = T // world
        t0 = rank * per                                    # this rank's tokens, as two micro-batches
        cuts = [(t0, t0 + per // 2), (t0 + per // 2, t0 + per)]
        probs = [dict(X=[p.X[a:b].to(dev) for a, b in cuts], dY=[p.dY[a:b].to(dev) for a, b in cuts],
                      W=p.W.to(dev).clone(), m=p.m.to(dev).clone(), v=p.v.to(dev).clone()) for p in ps]
        plan = dp.BucketPlan(SHAPES, 4 * 128 * 520, slots=2)
        pool = [torch.full((plan.slot_elems,), float("nan"), device=dev) for _ in range(plan.slots)]
        dp.bucket_step_adamw(probs, 3, HPT, plan, pool)                    # library kernels + NCCL all-reduce
        Bs = [dict(X=p.X[t0:t0 + per].to(dev), dY=p.dY[t0:t0 + per].to(dev), m=p.m.to(dev).clone()) for p in ps]
        dp.reduce_into_state(Bs, 0.9)
        torch.cuda.synchronize()
        out = [(_bits(d["W"]), d["m"].cpu().numpy(), d["v"].cpu().numpy(), b["m"].cpu().numpy()) for d, b in zip(probs, Bs)]
        parts = [None] * world
        dist.all_gather_object(parts, out)
        if rank == 0:
            q.put(parts)
    finally:
        dist.destroy_process_group()


def test_bucket_schedule_and_reduce_into_state_world2_nccl_match_the_all_token_oracle():
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs in one box")
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    parts = q.get()
    for pr in procs:
        pr.join(120)
        assert pr.exitcode == 0
    for i, p in enumerate(_problems()):
        (W0, m0, v0, B0), (W1, m1, v1, B1) = parts[0][i], parts[1][i]
        assert np.array_equal(W0, W1) and np.array_equal(m0, m1) and np.array_equal(v0, v1) and np.array_equal(B0, B1)
        G, E = fo.wgrad(_bits(p.dY), _bits(p.X), with_abs=True)
        Wb, m, v = _bits(p.W).copy(), p.m.numpy().copy(), p.v.numpy().copy()
        fo.adamw_fp32(Wb, m, v, G, 3, *HPT)
        d = 2.0 ** -21 * E + T * 2.0 ** -23 * E            # fp32 partial sums of four micro-batches + their accumulation
        assert (np.abs(m0.astype(np.float64) - m) <= (1 - HP["beta1"]) * d + 1e-4 * np.abs(m)).all()
        assert (np.abs(v0.astype(np.float64) - v) <= (1 - HP["beta2"]) * (2 * np.abs(G) * d + d * d) + 1e-4 * v).all()
        dW = np.abs(fo.bf16_to_f64(W0) - fo.bf16_to_f64(Wb))
        assert float((W0 == Wb).mean()) > 0.99 and (dW <= 2.0 ** -7 * np.abs(fo.bf16_to_f64(Wb)) + 2 * HP["lr"]).all()
        B = p.m.numpy().copy()
        fo.accumulate(B, G, 0.9)
        assert (np.abs(B0.astype(np.float64) - B) <= d + 2.0 ** -20 * np.abs(B)).all()

"""Data-parallel schedules of dp.py on CPU (gloo, world_size 2): SURVEY.md 8(f) rank 4 (302-304).

No GPU here, so the three injectable steps (wgrad into the bucket, update from the bucket, accumulate into state) are
supplied by the oracle; what is under test is dp.py itself: the bucket cutting, the slot rotation and its ordering, the
micro-batch accumulation, the all-reduce placement and the zero seed of reduce-into-state.  The result must be the
single-process oracle step on ALL tokens (Prop. 2(ii): the update sees the complete gradient), and the replicas must
stay bitwise in sync."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import dp, synth

SHAPES = [(384, 256), (200, 264)]
T = 96
HP = synth.HP_DEFAULT
HPT = (HP["lr"], HP["beta1"], HP["beta2"], HP["eps"], HP["wd"])


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_bucket_plan_covers_every_row_once_aligned_and_bounded():
    layer = [(4096, 4096), (1024, 4096), (1024, 4096), (4096, 4096), (14336, 4096), (14336, 4096), (4096, 14336)]
    for shapes, nbytes in ((layer, 256 << 20), (layer, 64 << 20), (SHAPES, 1), (SHAPES, 4 * 128 * 520), ([(128256, 4096)], 256 << 20)):
        plan = dp.BucketPlan(shapes, nbytes)
        seen = {p: 0 for p in range(len(shapes))}
        for bucket in plan.buckets:
            off = 0
            for pc in bucket:                              # pieces in order, packed back to back, rows contiguous per problem
                assert pc.offset == off and pc.r0 == seen[pc.p] and pc.r0 % dp.ROW_ALIGN == 0 and pc.r1 > pc.r0
                assert pc.cols == shapes[pc.p][1]
                seen[pc.p] = pc.r1
                off += pc.elems
            assert off <= plan.capacity_elems and off <= plan.slot_elems
        assert all(seen[p] == shapes[p][0] for p in seen)
        assert plan.transient_bytes == 2 * plan.slot_elems * 4
    # the transient does not grow with the model: 32 layers cut exactly like one
    assert dp.BucketPlan(layer * 32, 256 << 20).transient_bytes == dp.BucketPlan(layer, 256 << 20).transient_bytes
    with pytest.raises(ValueError):
        dp.BucketPlan(layer, 1 << 20, slots=0)


def _bits(t):
    return np.ascontiguousarray(synth.bf16_bits(t))


def _oracle_wgrad(pieces, first):
    for q in pieces:
        g = torch.from_numpy(fo.wgrad(_bits(q["dY"]), _bits(q["X"])).astype(np.float32))
        if first:
            q["m"].copy_(g)
        else:
            q["m"].add_(g)


def _oracle_update(G2d, state, step, hp):
    Wb, m, v = _bits(state["W"]).copy(), state["m"].numpy().copy(), state["v"].numpy().copy()
    fo.adamw_fp32(Wb, m, v, G2d.numpy().astype(np.float64), step, *hp)
    state["W"].copy_(torch.from_numpy(Wb.view(np.int16)).view(torch.bfloat16))
    state["m"].copy_(torch.from_numpy(m))
    state["v"].copy_(torch.from_numpy(v))


def _oracle_accumulate(problems, mu, state_dtype):
    for q in problems:
        B = q["m"].numpy().copy()
        fo.accumulate(B, fo.wgrad(_bits(q["dY"]), _bits(q["X"])), mu)
        q["m"].copy_(torch.from_numpy(B))


def _problems():
    return [synth.make_problem(f"p{i}", T, o, c, 300 + i) for i, (o, c) in enumerate(SHAPES)]


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ps = _problems()                                   # same seeds: the replicas start identical
        per = T // world
        t0 = rank * per                                    # this rank's tokens, as two micro-batches
        cuts = [(t0, t0 + per // 2), (t0 + per // 2, t0 + per)]
        probs = [dict(X=[p.X[a:b] for a, b in cuts], dY=[p.dY[a:b] for a, b in cuts], W=p.W.clone(), m=p.m.clone(),
                      v=p.v.clone()) for p in ps]
        plan = dp.BucketPlan(SHAPES, 4 * 128 * 520, slots=2)           # 128 rows of both problems per bucket
        assert len(plan.buckets) >= 3 and any(len(b) > 1 for b in plan.buckets)
        pool = [torch.full((plan.slot_elems,), float("nan")) for _ in range(plan.slots)]
        dp.bucket_step_adamw(probs, 3, HPT, plan, pool, wgrad=_oracle_wgrad, update=_oracle_update)
        # reduce-into-state: B replicated, mu on rank 0 only
        Bs = [dict(X=p.X[t0:t0 + per], dY=p.dY[t0:t0 + per], m=p.m.clone()) for p in ps]
        dp.reduce_into_state(Bs, 0.9, accumulate=_oracle_accumulate)
        out = [(_bits(d["W"]), d["m"].numpy(), d["v"].numpy(), b["m"].numpy()) for d, b in zip(probs, Bs)]
        parts = [None] * world
        dist.all_gather_object(parts, out)
        if rank == 0:
            q.put(parts)
    finally:
        dist.destroy_process_group()


def test_bucket_schedule_and_reduce_into_state_world2_match_the_all_token_oracle():
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
        # replicas in sync, bit for bit (every rank updates from the same reduced bucket)
        assert np.array_equal(W0, W1) and np.array_equal(m0, m1) and np.array_equal(v0, v1) and np.array_equal(B0, B1)
        # and equal to ONE oracle step on all T tokens; the bucket holds fp32 partial sums (4 of them), hence the slack
        G, E = fo.wgrad(_bits(p.dY), _bits(p.X), with_abs=True)
        Wb, m, v = _bits(p.W).copy(), p.m.numpy().copy(), p.v.numpy().copy()
        fo.adamw_fp32(Wb, m, v, G, 3, *HPT)
        d = 2.0 ** -21 * E                                  # four fp32-rounded partial sums and their fp32 additions
        assert (np.abs(m0.astype(np.float64) - m) <= (1 - HP["beta1"]) * d + 2.0 ** -22 * np.abs(m)).all()
        assert (np.abs(v0.astype(np.float64) - v) <= (1 - HP["beta2"]) * (2 * np.abs(G) * d + d * d) + 2.0 ** -22 * v).all()
        dW = np.abs(fo.bf16_to_f64(W0) - fo.bf16_to_f64(Wb))
        assert float((W0 == Wb).mean()) > 0.999 and (dW <= 2.0 ** -7 * np.abs(fo.bf16_to_f64(Wb)) + 2 * HP["lr"]).all()
        assert not np.array_equal(Wb, _bits(p.W))
        B = p.m.numpy().copy()
        fo.accumulate(B, G, 0.9)
        assert (np.abs(B0.astype(np.float64) - B) <= d + 2.0 ** -21 * np.abs(B)).all()

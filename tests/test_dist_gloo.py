"""N > 1 host logic on CPU (gloo, world_size 2): the path shards along the weight with no collective
(Prop. 2(i)); each rank's row shard, computed alone, must be bit-identical to the same
rows of the unsharded result.  No GPU here, so each rank evaluates its shard with the oracle --
what is under test is the sharding / gathering / timing-reduction logic of shard.py."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import shard, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_rows_partitions_and_aligns():
    for out in (8, 128, 384, 1024, 4096, 14336, 128256):
        for world in (1, 2, 3, 4, 8):
            spans = [shard.shard_rows(out, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == out
            for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
                assert a1 == b0 and a0 <= a1
            assert all(a0 % shard.ROW_ALIGN == 0 for a0, a1 in spans if a1 > a0)
            sizes = [a1 - a0 for a0, a1 in spans]
            assert max(sizes) - min(sizes) <= shard.ROW_ALIGN or out < world * shard.ROW_ALIGN
    with pytest.raises(ValueError):
        shard.shard_rows(128, 2, 2)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        hp = synth.HP_DEFAULT
        p = synth.make_problem("t", 96, 384, 256, 77)          # same seed on every rank
        d = dict(X=p.X, dY=p.dY, W=p.W.clone(), m=p.m.clone(), v=p.v.clone())
        s = shard.shard_problem(d, world, rank)
        r0, r1 = s["rows"]
        Wb = synth.bf16_bits(s["W"]).copy()
        m = s["m"].numpy().copy()
        v = s["v"].numpy().copy()
        G = fo.wgrad(synth.bf16_bits(s["dY"]), synth.bf16_bits(s["X"]))
        fo.adamw_fp32(Wb, m, v, G, 3, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
        # gather the shards (test plumbing only -- the data path itself has no collective)
        parts = [None] * world
        dist.all_gather_object(parts, (r0, r1, Wb, m, v))
        tmax = shard.max_over_ranks(10.0 + rank)
        if rank == 0:
            q.put((parts, tmax))
    finally:
        dist.destroy_process_group()


def test_row_sharded_update_equals_unsharded_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    parts, tmax = q.get()
    for pr in procs:
        pr.join(120)
        assert pr.exitcode == 0
    assert tmax == 11.0                                   # slowest rank's time
    hp = synth.HP_DEFAULT
    p = synth.make_problem("t", 96, 384, 256, 77)
    Wb = synth.bf16_bits(p.W).copy()
    m, v = p.m.numpy().copy(), p.v.numpy().copy()
    G = fo.wgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.X))
    fo.adamw_fp32(Wb, m, v, G, 3, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    covered = 0
    for r0, r1, Ws, ms, vs in sorted(parts, key=lambda t: t[0]):
        assert r0 == covered
        covered = r1
        assert np.array_equal(Ws, Wb[r0:r1]) and np.array_equal(ms, m[r0:r1]) and np.array_equal(vs, v[r0:r1])
    assert covered == 384


def test_shard_problem_views_alias_the_state():
    p = synth.make_problem("t", 16, 256, 512, 5)
    d = dict(X=p.X, dY=p.dY, W=p.W, m=p.m, v=p.v,
             m_scale=torch.zeros(256, 2), v_scale=torch.zeros(256, 2))
    s = shard.shard_problem(d, 2, 1)
    assert s["rows"] == (128, 256)
    assert s["W"].data_ptr() == p.W[128:].data_ptr() and s["m_scale"].shape == (128, 2)
    # dY is a column-slice VIEW (row pitch = the full out, passed to the ABI as lddy), not a copy
    assert s["dY"].shape == (16, 128) and s["dY"].stride() == (256, 1) and s["dY"].data_ptr() == p.dY[:, 128:].data_ptr()
    assert shard.shard_problem(d, 4, 3) is None           # 2 row blocks over 4 ranks: ranks 2,3 empty

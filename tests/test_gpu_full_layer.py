"""GPU parity at FULL size, every row: the configs[1] / configs[2] grouped launch (the configuration bench.py times)
against the oracle element by element on every row of every projection, >= 1/16 of the rows of gate_proj at
T = 2048 / 8192 (ring and direct dispatch paths) spread over all waves, and the edge cases include/forge.h promises
(NaN / Inf propagation, an all-zero int8 block inside a full tile, the decay-only step dY = 0 of PAPER.md:292)."""
import numpy as np
import pytest
import torch

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import binding as fb
from paper_2606_22932_b200 import synth
import parity_util as pu
from test_gpu_parity import DEV, HP, compare, gpu_state, hp_args, oracle_step

pytestmark = pytest.mark.gpu
ROW_CHUNK = 512


@pytest.mark.parametrize("moment", ["fp32", "bf16", "int8"])
def test_config1_2_whole_layer_every_row_against_the_oracle(moment):
    """All 218 103 808 weight elements of the Llama-3.1-8B layer, one grouped launch, compared with the oracle row
    chunk by row chunk (rows are independent; chunks only bound the host memory of the fp64 gradient)."""
    layer = synth.make_layer(512, seed=synth.BASE_SEED + 1)
    pairs = [gpu_state(p, moment) for p in layer]
    ds = [d for d, _ in pairs]
    before = fb.forge_launch_count()
    fb.forge_wgrad_adamw_grouped(ds, 10, *pu.hp_tuple(HP), {"fp32": 0, "bf16": 1, "int8": 2}[moment])
    torch.cuda.synchronize()
    assert fb.forge_launch_count() - before == 1
    stats = dict(n=0, w_equal=0, m_code_equal=0, v_code_equal=0)
    for p, (d, o) in zip(layer, pairs):
        host = {k: pu.to_np(d[k]) for k in d if k not in ("X", "dY")}        # one D2H per tensor
        for r0 in range(0, p.out, ROW_CHUNK):
            rows = (r0, min(p.out, r0 + ROW_CHUNK))
            ref, G, E = oracle_step(o, moment, 10, rows)
            view = {k: host[k][rows[0]:rows[1]] for k in host}
            compare_host(view, ref, G, E, 512, moment, f"{moment} {p.name} rows {rows}", o["W"][rows[0]:rows[1]])
            stats["n"] += G.size
            stats["w_equal"] += int((view["W"] == ref["W"]).sum())
            if moment == "int8":
                stats["m_code_equal"] += int((view["m"] == ref["m"]).sum())
                stats["v_code_equal"] += int((view["v"] == ref["v"]).sum())
    pu.record("whole_layer", moment=moment, elements=stats["n"], w_bit_identical=stats["w_equal"] / stats["n"],
              m_code_identical=stats["m_code_equal"] / stats["n"] if moment == "int8" else None,
              v_code_identical=stats["v_code_equal"] / stats["n"] if moment == "int8" else None)
    assert stats["n"] == 218103808


def compare_host(view, ref, G, E, T, moment, label, W_prev):
    """test_gpu_parity.compare on host arrays already copied back."""
    tol = pu.Tol(G.shape)
    e = tol.step(G, E, T, HP)
    wprop = ref.get("_wprop", 0.0)
    if moment == "int8":
        pu.check_int8(view["W"], view["m"], view["v"], view["m_scale"], view["v_scale"], ref["W"], ref["m"], ref["v"],
                      ref["m_scale"], ref["v_scale"], G, e, HP, label, W_prev=W_prev, w_prop=wprop)
    else:
        pu.check_fp(view["W"], view["m"], view["v"], ref["W"], ref["m"], ref["v"], G, e, tol, HP, moment, label, W_prev=W_prev,
                    w_prop=wprop)


@pytest.mark.parametrize("T", [2048, 8192])
def test_config3_gate_one_sixteenth_of_the_rows_spread_over_all_waves(T):
    """configs[3] at T = 2048 (large-T ring path) and T = 8192 (direct state path): 7 x 128 rows = 1/16 of gate_proj,
    from the first tile to the last partial wave."""
    p = synth.make_problem("gate", T, 14336, 4096, seed=synth.BASE_SEED + 3)
    d, o = gpu_state(p, "fp32")
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 10, **HP)
    torch.cuda.synchronize()
    ranges = pu.spread_rows(14336, 16, 128)
    assert sum(b - a for a, b in ranges) * 16 >= 14336 and ranges[0][0] == 0 and ranges[-1][1] == 14336
    for rows in ranges:
        ref, G, E = oracle_step(o, "fp32", 10, rows)
        compare(d, ref, G, E, T, "fp32", rows, label=f"gate T={T} rows {rows}", W_prev=o["W"])


def test_fp8_and_sr_whole_layer_every_row_against_the_oracle():
    """The two other storage decisions of SURVEY.md 8(f) rank 1 at full size, every row: e4m3 moments with delayed
    scaling (codes within one e4m3 step of the oracle's fp64 `e4m3(x/s)`, > 99 % identical, amax to 1e-4) and the
    stochastic-rounding store (W always a bf16 neighbour of the oracle's choice, > 99.5 % equal; reading S16 / S17).
    The measured agreement rates go to gpurun_out/parity_stats.jsonl."""
    hpt = pu.hp_tuple(HP)
    layer = synth.make_layer(512, seed=synth.BASE_SEED + 1)
    # ---- fp8
    devs, keep = [], []
    for p in layer:
        mq, ms = fo.fp8_quantize(p.m.numpy())
        vq, vs = fo.fp8_quantize(p.v.numpy())
        keep.append((mq, ms, vq, vs))
        devs.append(dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=torch.from_numpy(mq.copy()).to(DEV),
                         v=torch.from_numpy(vq.copy()).to(DEV), m_scale=torch.from_numpy(ms.copy()).to(DEV),
                         v_scale=torch.from_numpy(vs.copy()).to(DEV)))
    fb.forge_wgrad_adamw_grouped(devs, 10, *hpt, fb.FP8)
    torch.cuda.synchronize()
    n = same_w = same_m = same_v = 0
    for p, d, (mq, ms, vq, vs) in zip(layer, devs, keep):
        dYb, Xb = synth.bf16_bits(p.dY), synth.bf16_bits(p.X)
        Wg, mg, vg = synth.bf16_bits(d["W"]), d["m"].cpu().numpy(), d["v"].cpu().numpy()
        Wall = synth.bf16_bits(p.W)
        amax_m = amax_v = 0.0
        for r0 in range(0, p.out, ROW_CHUNK):
            r1 = min(p.out, r0 + ROW_CHUNK)
            G = fo.wgrad(dYb, Xb, rows=(r0, r1))
            Wo, mo, vo, mso, vso = Wall[r0:r1].copy(), mq[r0:r1].copy(), vq[r0:r1].copy(), ms.copy(), vs.copy()
            fo.adamw_fp8(Wo, mo, vo, mso, vso, G, 10, *hpt)
            amax_m, amax_v = max(amax_m, float(mso[1])), max(amax_v, float(vso[1]))
            for got, ref in ((mg[r0:r1], mo), (vg[r0:r1], vo)):
                assert np.abs((got & 0x7F).astype(int) - (ref & 0x7F).astype(int)).max() <= 1, (p.name, r0)
            n += G.size
            same_w += int((Wg[r0:r1] == Wo).sum()); same_m += int((mg[r0:r1] == mo).sum()); same_v += int((vg[r0:r1] == vo).sum())
        assert abs(float(d["m_scale"].cpu()[1]) - amax_m) <= 1e-4 * amax_m and abs(float(d["v_scale"].cpu()[1]) - amax_v) <= 1e-4 * amax_v
    pu.record("whole_layer_fp8", elements=n, w_bit_identical=same_w / n, m_code_identical=same_m / n, v_code_identical=same_v / n)
    assert n == 218103808 and same_w / n > 0.99 and same_m / n > 0.99 and same_v / n > 0.99
    del devs
    # ---- stochastic-rounding store (fp32 moments), whole projections (the generator is keyed on the global row / column)
    probs = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in layer]
    seed = (11 << 40) + 2026
    fb.forge_wgrad_adamw_sr_grouped(probs, 10, *hpt, fb.FP32, seed)
    torch.cuda.synchronize()
    n = same = 0
    for i, (p, d) in enumerate(zip(layer, probs)):
        W0 = synth.bf16_bits(p.W)
        Wo, mo, vo = W0.copy(), p.m.numpy().copy(), p.v.numpy().copy()
        dYb, Xb = synth.bf16_bits(p.dY), synth.bf16_bits(p.X)
        G, E = fo.wgrad(dYb, Xb, with_abs=True)
        fo.adamw_fp32_sr(Wo, mo, vo, G, 10, *hpt, seed=seed, stream=i)
        Wg = synth.bf16_bits(d["W"])
        # the GPU's choice and the oracle's are both bf16 neighbours of (nearly) the same W': at most one bf16 step
        # apart, plus the reading-T1 terms where W' cancels to ~0 (a handful of elements per projection)
        far = np.abs(Wg.astype(np.int32) - Wo.astype(np.int32)) > 1
        for r, c in np.argwhere(far)[:64]:
            r0, r1 = int(r), int(r) + 1
            e = 512 * 2.0 ** -23 * E[r0:r1]
            wprop = pu.w_propagated("fp32", W0[r0:r1].copy(), p.m.numpy()[r0:r1].copy(), p.v.numpy()[r0:r1].copy(), G[r0:r1], e, 10, HP)
            Wr = fo.bf16_to_f64(Wo[r0:r1])
            bound = 2 * pu.bf16_ulp(Wr) + pu.fp32_eval_err(W0[r0:r1], Wr) + wprop
            assert abs(fo.bf16_to_f64(Wg[r0:r1])[0, c] - Wr[0, c]) <= bound[0, c], (p.name, int(r), int(c))
        assert int(far.sum()) <= 64 and far.mean() < 1e-6, (p.name, int(far.sum()))
        n += Wo.size
        same += int((Wg == Wo).sum())
        del G, E
    pu.record("whole_layer_sr", elements=n, w_equal_to_oracle_choice=same / n)
    assert same / n > 0.995


def test_layer_backward_full_llama_layer_dgrad_and_update_against_the_oracle():
    """forge_layer_backward_grouped on the whole cfg-1 layer (the configuration bench.py's `layer_backward` leg times):
    one dgrad launch over 304 pair-tiles of depth 1024 ... 14336 in the longest-first order, then the fused launch.
    Every dX element against the oracle's fp64 dY.W from the PRE-update weights; W, m, v bit-identical to the plain
    grouped call (whose own parity is the test above)."""
    layer = synth.make_layer(512, seed=synth.BASE_SEED + 1)
    probs = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in layer]
    twins = [dict(X=d["X"], dY=d["dY"], W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p, d in zip(layer, probs)]
    dXs = [torch.full((p.T, p.inn), float("nan"), dtype=torch.bfloat16, device=DEV) for p in layer]
    n0 = fb.forge_launch_count()
    fb.forge_layer_backward_grouped(probs, dXs, *hp_args(10), fb.FP32)
    assert fb.forge_launch_count() - n0 == 2
    fb.forge_wgrad_adamw_grouped(twins, *hp_args(10), fb.FP32)
    torch.cuda.synchronize()
    for p, d, t, dX in zip(layer, probs, twins, dXs):
        for k in ("W", "m", "v"):
            assert torch.equal(d[k], t[k]), (p.name, k)
        dYf, Wf = fo.bf16_to_f64(synth.bf16_bits(p.dY)), fo.bf16_to_f64(synth.bf16_bits(p.W))
        ref = fo.dgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.W))
        got = fo.bf16_to_f64(synth.bf16_bits(dX))
        bound = p.out * 2.0 ** -23 * (np.abs(dYf) @ np.abs(Wf))
        bad = np.abs(got - ref) > pu.bf16_ulp(ref) + bound
        assert not bad.any(), (p.name, int(bad.sum()), float(np.abs(got - ref).max()))
        exact = float((synth.bf16_bits(dX) == fo.f64_to_bf16(ref)).mean())
        pu.record("dgrad_layer", name=p.name, dx_bit_identical=exact)
        assert exact > 0.98, (p.name, exact)


# ------------------------------------------------------------------------------ edge cases ---
def test_nan_and_inf_propagate_to_exactly_the_affected_row_and_column():
    """include/forge.h: "NaN/Inf in the inputs propagate by IEEE rules (to the rows / columns of G they enter and
    nowhere else)".  A NaN in dY[t, p] poisons row p of G, an Inf in X[t, q] column q (and NaN where it meets a
    zero-sign cancellation); everything else must be bit-identical to the clean run."""
    p = synth.make_problem("n", 300, 384, 768, seed=901)
    clean, _ = gpu_state(p, "fp32")
    fb.forge_wgrad_adamw(clean["X"], clean["dY"], clean["W"], clean["m"], clean["v"], 7, **HP)
    d, _ = gpu_state(p, "fp32")
    pr, qc = 200, 515                                    # second 128-row block; third 256-column tile... col 515 of 768
    d["dY"][17, pr] = float("nan")
    d["X"][250, qc] = float("inf")
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 7, **HP)
    torch.cuda.synchronize()
    touched = torch.zeros(384, 768, dtype=torch.bool, device=DEV)
    touched[pr, :] = True
    touched[:, qc] = True
    for k in ("W", "m", "v"):
        a, b = d[k].float(), clean[k].float()
        assert torch.equal(d[k][~touched], clean[k][~touched]), f"{k}: poison leaked outside row {pr} / column {qc}"
        assert torch.isnan(a[pr, :]).all(), f"{k}: row {pr} must be NaN"
        col = a[:, qc]
        assert (~torch.isfinite(col)).all(), f"{k}: column {qc} must be Inf or NaN"
        assert torch.isfinite(b).all()


def test_dy_zero_is_the_decay_only_step():
    """PAPER.md:292 Remark 1: G = 0 gives m' = b1 m, v' = b2 v and W' from those (the decay-only step); against the
    oracle on every element, and W moves by decay + the stale-moment update only."""
    p = synth.make_problem("z", 256, 384, 512, seed=902)
    p.dY.zero_()
    for moment in ("fp32", "int8"):
        d, o = gpu_state(p, moment)
        fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 10, m_scale=d.get("m_scale"), v_scale=d.get("v_scale"), **HP)
        torch.cuda.synchronize()
        ref, G, E = oracle_step(o, moment, 10)
        assert not G.any() and not E.any()
        compare(d, ref, G, E, 256, moment, label=f"dY=0 {moment}", W_prev=o["W"])
        if moment == "fp32":
            b1 = np.float64(np.float32(HP["beta1"]))
            assert np.allclose(pu.to_np(d["m"]), b1 * p.m.numpy().astype(np.float64), rtol=1e-6, atol=0)


def test_all_zero_int8_block_inside_a_full_tile():
    """App. B / reading S6: a block whose new moments are all zero stores a = 0 and codes 0 (no division by the
    scale); here rows 130..133 x columns 256..511 of a multi-tile problem have zero state AND zero gradient (their dY
    columns are zero), in the middle of blocks that are busy."""
    p = synth.make_problem("q", 200, 384, 768, seed=903)
    p.dY[:, 130:134] = 0
    p.m[130:134, 256:512] = 0
    p.v[130:134, 256:512] = 0
    d, o = gpu_state(p, "int8")
    assert not o["m_scale"][130:134, 1].any() and not o["v_scale"][130:134, 1].any()
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 10, m_scale=d["m_scale"], v_scale=d["v_scale"], **HP)
    torch.cuda.synchronize()
    ref, G, E = oracle_step(o, "int8", 10)
    compare(d, ref, G, E, 200, "int8", label="zero block", W_prev=o["W"])
    assert not d["m"][130:134, 256:512].any() and not d["v"][130:134, 256:512].any()
    assert not d["m_scale"][130:134, 1].any() and not d["v_scale"][130:134, 1].any()
    assert torch.isfinite(d["W"].float()).all()
    # the same rows' OTHER blocks carry state (zero gradient there too: pure decay of the codes)
    assert d["m_scale"][130:134, 0].all() and d["v_scale"][130:134, 2].all()


@pytest.mark.parametrize("hp_over, label", [
    (dict(lr=0.0), "lr = 0"),                       # no step: W' = (1 - 0) W bit for bit, moments still move
    (dict(lr=1e-30, wd=0.0), "lr = 1e-30"),         # a huge but finite folded denominator
    (dict(lr=1e-44, wd=0.0), "lr = 1e-44"),         # subnormal lr: c / step leaves the fp32 range, the no-step constants take over
    (dict(lr=1.0, wd=0.0), "lr = 1"),               # the largest step size the folded denominator sees
    (dict(eps=0.0), "eps = 0"),                     # the denominator is sqrt(v_hat) alone (v' > 0 everywhere here)
    (dict(eps=1e-3, beta1=0.0), "eps = 1e-3, beta1 = 0"),
])
def test_step_size_folded_into_the_denominator_edge_hyperparameters(hp_over, label):
    """The kernels evaluate W' = decay W + m' * rcp(-(sqrt(v') c + eps) / step) (adamw_math.cuh): the hyper-parameter
    corners of that folding -- no step at all, a step too small for fp32, a large one, eps = 0 -- against the oracle's
    plain Alg. 1 lines 9-10, fp32 and int8 moments, steps 1 and 50."""
    hp = dict(HP, **hp_over)
    p = synth.make_problem("h", 200, 384, 768, seed=910)
    for moment in ("fp32", "int8"):
        for step in (1, 50):
            d, o = gpu_state(p, moment)
            W0 = d["W"].clone()
            fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], step, m_scale=d.get("m_scale"),
                                 v_scale=d.get("v_scale"), **hp)
            torch.cuda.synchronize()
            G, E = fo.wgrad(o["dY"], o["X"], with_abs=True)
            W, m, v = o["W"].copy(), o["m"].copy(), o["v"].copy()
            tol = pu.Tol(G.shape)
            e = tol.step(G, E, 200, hp)
            args = (step,) + pu.hp_tuple(hp)
            if moment == "fp32":
                wprop = pu.w_propagated("fp32", W, m, v, G, e, step, hp)
                fo.adamw_fp32(W, m, v, G, *args)
                pu.check_fp(pu.to_np(d["W"]), pu.to_np(d["m"]), pu.to_np(d["v"]), W, m, v, G, e, tol, hp, "fp32",
                            f"{label} fp32 step {step}", W_prev=o["W"], w_prop=wprop)
            else:
                ms, vs = o["m_scale"].copy(), o["v_scale"].copy()
                wprop = pu.w_propagated("int8", W, m, v, G, e, step, hp, (ms, vs))
                fo.adamw_int8(W, m, v, ms, vs, G, *args)
                pu.check_int8(pu.to_np(d["W"]), pu.to_np(d["m"]), pu.to_np(d["v"]), pu.to_np(d["m_scale"]),
                              pu.to_np(d["v_scale"]), W, m, v, ms, vs, G, e, hp, f"{label} int8 step {step}",
                              W_prev=o["W"], w_prop=wprop)
            assert torch.isfinite(d["W"].float()).all()
            if hp["lr"] < 1e-20:
                assert torch.equal(d["W"], W0), f"{label} {moment}: W must not move"

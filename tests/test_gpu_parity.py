"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
BASELINE.json configs 0-3 and the edge cases; tolerances from tests/parity_util.py."""
import os

import numpy as np
import pytest
import torch

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import binding as fb
from paper_2606_22932_b200 import synth
import parity_util as pu

pytestmark = pytest.mark.gpu
HP = synth.HP_DEFAULT
DEV = "cuda"


def hp_args(step):
    return (step,) + pu.hp_tuple(HP)


def gpu_state(p: synth.Problem, moment: str):
    """Device copies of one problem's tensors + the oracle-side numpy twins (same bits)."""
    d = dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone())
    o = dict(X=synth.bf16_bits(p.X), dY=synth.bf16_bits(p.dY), W=synth.bf16_bits(p.W).copy())
    if moment == "fp32":
        d["m"], d["v"] = p.m.to(DEV).clone(), p.v.to(DEV).clone()
        o["m"], o["v"] = p.m.numpy().copy(), p.v.numpy().copy()
    elif moment == "bf16":
        mb, vb = p.m.to(torch.bfloat16), p.v.to(torch.bfloat16)
        d["m"], d["v"] = mb.to(DEV), vb.to(DEV)
        o["m"], o["v"] = synth.bf16_bits(mb).copy(), synth.bf16_bits(vb).copy()
    else:  # int8: the oracle's quantiser produces the seeds for both sides (reading S8)
        mq, ms, vq, vs = fo.quantize(p.m.numpy(), p.v.numpy())
        o.update(m=mq, v=vq, m_scale=ms, v_scale=vs)
        d.update(m=torch.from_numpy(mq.copy()).to(DEV), v=torch.from_numpy(vq.copy()).to(DEV),
                 m_scale=torch.from_numpy(ms.copy()).to(DEV), v_scale=torch.from_numpy(vs.copy()).to(DEV))
    return d, o


def oracle_step(o, moment, step, rows=None):
    """Oracle on all rows or on a row range; returns (state after the step on those rows, G, E).  ref["_wprop"] is the
    accumulation-error bound of g carried through the update (parity_util.w_propagated)."""
    G, E = fo.wgrad(o["dY"], o["X"], rows=rows, with_abs=True)
    sl = slice(None) if rows is None else slice(*rows)
    W, m, v = o["W"][sl].copy(), o["m"][sl].copy(), o["v"][sl].copy()      # the seeds stay untouched
    e = o["X"].shape[0] * 2.0 ** -23 * E
    scales = (o["m_scale"][sl], o["v_scale"][sl]) if moment == "int8" else None
    wprop = pu.w_propagated(moment, W, m, v, G, e, step, HP, scales)
    if moment == "fp32":
        fo.adamw_fp32(W, m, v, G, *hp_args(step))
        return dict(W=W, m=m, v=v, _wprop=wprop), G, E
    if moment == "bf16":
        fo.adamw_bf16(W, m, v, G, *hp_args(step))
        return dict(W=W, m=m, v=v, _wprop=wprop), G, E
    ms, vs = o["m_scale"][sl].copy(), o["v_scale"][sl].copy()
    fo.adamw_int8(W, m, v, ms, vs, G, *hp_args(step))
    return dict(W=W, m=m, v=v, m_scale=ms, v_scale=vs, _wprop=wprop), G, E


def compare(d, ref, G, E, T, moment, rows=None, label="", W_prev=None):
    sl = slice(None) if rows is None else slice(*rows)
    W_prev = None if W_prev is None else W_prev[sl]
    tol = pu.Tol(G.shape)
    e = tol.step(G, E, T, HP)
    wprop = ref.get("_wprop", 0.0)
    g = {k: pu.to_np(d[k][sl]) for k in ref if not k.startswith("_")}
    if moment == "int8":
        pu.check_int8(g["W"], g["m"], g["v"], g["m_scale"], g["v_scale"], ref["W"], ref["m"], ref["v"],
                      ref["m_scale"], ref["v_scale"], G, e, HP, label, W_prev=W_prev, w_prop=wprop)
    else:
        pu.check_fp(g["W"], g["m"], g["v"], ref["W"], ref["m"], ref["v"], G, e, tol, HP, moment, label, W_prev=W_prev,
                    w_prop=wprop)


# ------------------------------------------------------------------------------ config 0 -----
def test_config0_three_chained_steps_fp32():
    """BASELINE.json cfg 0: W[384,256], T=128, zero state, fresh inputs per step, 3 steps."""
    W = synth.config0_weight()
    Wo, mo, vo = synth.bf16_bits(W).copy(), np.zeros((384, 256), np.float32), np.zeros((384, 256), np.float32)
    Wg, mg, vg = W.to(DEV), torch.zeros(384, 256, device=DEV), torch.zeros(384, 256, device=DEV)
    tol = pu.Tol((384, 256))
    for step in (1, 2, 3):
        X, dY = synth.config0_step_inputs(step)
        fb.forge_wgrad_adamw(X.to(DEV), dY.to(DEV), Wg, mg, vg, step, **HP)
        G, E = fo.wgrad(synth.bf16_bits(dY), synth.bf16_bits(X), with_abs=True)
        W_prev = Wo.copy()
        fo.adamw_fp32(Wo, mo, vo, G, *hp_args(step))
        e = tol.step(G, E, 128, HP)
        torch.cuda.synchronize()
        pu.check_fp(pu.to_np(Wg), pu.to_np(mg), pu.to_np(vg), Wo, mo, vo, G, e, tol, HP, "fp32", f"cfg0 step {step}",
                    W_prev=W_prev)


# ------------------------------------------------------------------------------ small shapes -
@pytest.mark.parametrize("moment", ["fp32", "bf16", "int8"])
@pytest.mark.parametrize("T,out,inn", [(512, 384, 768), (200, 136, 264), (1, 128, 256), (33, 8, 16), (2048, 256, 512)])
def test_small_shapes_full_compare(moment, T, out, inn):
    """Several tiles + ragged tails in every dimension (T not a multiple of the token chunk, out
    not a multiple of 128, in not a multiple of 256), T=1, tiny W, and the large-T kernel variant."""
    if moment == "int8" and inn % 256:
        inn = 512 if inn > 256 else 256
    p = synth.make_problem("t", T, out, inn, seed=100 + T + out)
    d, o = gpu_state(p, moment)
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 10, m_scale=d.get("m_scale"),
                         v_scale=d.get("v_scale"), **HP)
    torch.cuda.synchronize()
    ref, G, E = oracle_step(o, moment, 10)
    compare(d, ref, G, E, T, moment, label=f"{moment} T={T} {out}x{inn}", W_prev=o["W"])


# ------------------------------------------------------------------------------ configs 1, 2 -
@pytest.fixture(scope="module")
def layer_cpu():
    return synth.make_layer(512, seed=synth.BASE_SEED + 1)


@pytest.mark.parametrize("moment", ["fp32", "bf16", "int8"])
def test_config1_2_llama_layer_grouped_sampled_rows(layer_cpu, moment):
    """BASELINE.json cfg 1 (fp32) and cfg 2 (bf16, int8): the 7 projections of a Llama-3.1-8B layer
    at full size in ONE grouped launch (the configuration bench.py times); the oracle is exact on
    a deterministic sample of rows of every projection (rows are independent)."""
    ds, os_ = zip(*[gpu_state(p, moment) for p in layer_cpu])
    before = fb.forge_launch_count()
    fb.forge_wgrad_adamw_grouped(list(ds), 10, *pu.hp_tuple(HP), {"fp32": 0, "bf16": 1, "int8": 2}[moment])
    torch.cuda.synchronize()
    assert fb.forge_launch_count() - before == 1
    for p, d, o in zip(layer_cpu, ds, os_):
        for rows in pu.sample_rows(p.out):
            ref, G, E = oracle_step(o, moment, 10, rows)
            compare(d, ref, G, E, 512, moment, rows, label=f"{moment} {p.name} rows {rows}", W_prev=o["W"])


def test_config2_low_precision_moments_track_fp32_moments(layer_cpu):
    """cfg 2 'each compared against fp32 moments': one step from the same seeds, the bf16 and int8
    results stay within their storage resolution of the fp32-moment result (k projection)."""
    p = layer_cpu[1]
    res = {}
    for moment in ("fp32", "bf16", "int8"):
        d, _ = gpu_state(p, moment)
        fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 10, m_scale=d.get("m_scale"),
                             v_scale=d.get("v_scale"), **HP)
        res[moment] = d
    torch.cuda.synchronize()
    m32 = res["fp32"]["m"].double()
    mb = res["bf16"]["m"].double()
    m0 = p.m.to(DEV).double().abs()
    # bf16 seeds differ from the fp32 seeds by <= 2^-9 |m0|, the bf16 store adds <= 2^-9 |m'|
    assert ((mb - m32).abs() <= 2.0 ** -8 * (m0 + m32.abs()) + 1e-12).all()
    mq = fo.dequantize_m(pu.to_np(res["int8"]["m"]), pu.to_np(res["int8"]["m_scale"]))
    s = np.repeat(pu.to_np(res["int8"]["m_scale"]).astype(np.float64) / 127, 256, 1)
    assert (np.abs(mq - m32.cpu().numpy()) <= 1.01 * s).all()       # old + new quantisation step
    w32 = res["fp32"]["W"].double()
    for k in ("bf16", "int8"):
        assert ((res[k]["W"].double() - w32).abs() <= 4 * HP["lr"]).all()


# ------------------------------------------------------------------------------ config 3 -----
@pytest.mark.parametrize("T", [512, 2048, 8192])
def test_config3_gate_proj_token_sweep_sampled_rows(T):
    """BASELINE.json cfg 3: gate_proj W[14336,4096], fp32 moments, T in {512, 2048, 8192}."""
    p = synth.make_problem("gate", T, 14336, 4096, seed=synth.BASE_SEED + 3)
    d, o = gpu_state(p, "fp32")
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 10, **HP)
    torch.cuda.synchronize()
    for rows in pu.sample_rows(14336, n_ranges=2, width=4):
        ref, G, E = oracle_step(o, "fp32", 10, rows)
        compare(d, ref, G, E, T, "fp32", rows, label=f"gate T={T} rows {rows}", W_prev=o["W"])


# ------------------------------------------------------------------------------ exactness ----
@pytest.mark.parametrize("moment", ["fp32", "bf16", "int8"])
@pytest.mark.parametrize("T", [512, 2048])
def test_fused_equals_store_g_twin_plus_same_update_bitwise(moment, T):
    """PAPER.md:294 / gate T0 ('max dW = 0'): the fused kernel vs the store-G twin
    followed by the same per-element update must be bit-identical."""
    p = synth.make_problem("x", T, 640, 768, seed=7)
    d1, _ = gpu_state(p, moment)
    d2 = {k: v.clone() for k, v in d1.items()}
    fb.forge_wgrad_adamw(d1["X"], d1["dY"], d1["W"], d1["m"], d1["v"], 5, m_scale=d1.get("m_scale"),
                         v_scale=d1.get("v_scale"), **HP)
    G = torch.full((640, 768), float("nan"), device=DEV)
    fb.forge_wgrad_store_g(d2["X"], d2["dY"], G)
    assert not torch.isnan(G).any()
    fb.forge_adamw_from_g(G, d2["W"], d2["m"], d2["v"], 5, m_scale=d2.get("m_scale"), v_scale=d2.get("v_scale"), **HP)
    torch.cuda.synchronize()
    for k in d1:
        assert torch.equal(d1[k].view(torch.uint8), d2[k].view(torch.uint8)), f"{moment}: {k} differs from the unfused twin"


@pytest.mark.parametrize("moment", ["fp32", "bf16"])
@pytest.mark.parametrize("out,inn", [(640, 768), (600, 528), (200, 264)])
def test_direct_state_path_at_large_T_equals_store_g_twin_bitwise(moment, out, inn):
    """T >= 8192 takes the ring-less direct epilogue (32-byte global accesses, thread = row) when every row is a
    whole number of 16-column vectors; (200, 264) is not and falls back to the TMA ring.  Ragged row blocks, several
    column tiles; bit-identical to the store-G twin plus the same update either way."""
    p = synth.make_problem("x", 8192, out, inn, seed=17)
    d1, _ = gpu_state(p, moment)
    d2 = {k: v.clone() for k, v in d1.items()}
    fb.forge_wgrad_adamw(d1["X"], d1["dY"], d1["W"], d1["m"], d1["v"], 5, **HP)
    G = torch.empty(out, inn, device=DEV)
    fb.forge_wgrad_store_g(d2["X"], d2["dY"], G)
    fb.forge_adamw_from_g(G, d2["W"], d2["m"], d2["v"], 5, **HP)
    torch.cuda.synchronize()
    for k in d1:
        assert torch.equal(d1[k].view(torch.uint8), d2[k].view(torch.uint8)), f"{moment}: {k} differs from the unfused twin"
    assert not torch.equal(d1["W"], p.W.to(DEV))


@pytest.mark.parametrize("moment", ["fp32", "int8"])
def test_strided_operand_views_fused_qkv_bitwise_and_dgrad(moment):
    """ldx / lddy (include/forge.h): q, k, v read column slices of ONE fused dY[T, 512+256+256] and a column slice of a
    wider X; the result must be bit-identical to the same call on dense copies of the slices, and the dgrad of
    forge_layer_backward_grouped must read the strided dY too."""
    T, inn, outs = 200, 512, (512, 256, 256)
    wide_x = torch.randn(T, inn + 64, generator=torch.Generator().manual_seed(5)).to(torch.bfloat16).to(DEV)
    fused_dy = (torch.randn(T, sum(outs), generator=torch.Generator().manual_seed(6)) * 1e-2).to(torch.bfloat16).to(DEV)
    X = wide_x[:, 32:32 + inn]
    views, dense, c0 = [], [], 0
    for i, o in enumerate(outs):
        p = synth.make_problem(f"p{i}", T, o, inn, seed=30 + i)
        d, _ = gpu_state(p, moment)
        dY = fused_dy[:, c0:c0 + o]
        c0 += o
        views.append(dict(d, X=X, dY=dY))
        dense.append({k: v.clone() for k, v in dict(d, X=X.contiguous(), dY=dY.contiguous()).items()})
    assert not views[1]["dY"].is_contiguous() and not X.is_contiguous()
    mdt = {"fp32": fb.FP32, "int8": fb.INT8}[moment]
    dXv = [torch.empty(T, inn, dtype=torch.bfloat16, device=DEV) for _ in outs]
    dXd = [torch.empty(T, inn, dtype=torch.bfloat16, device=DEV) for _ in outs]
    fb.forge_layer_backward_grouped(views, dXv, *hp_args(7), mdt)
    fb.forge_layer_backward_grouped(dense, dXd, *hp_args(7), mdt)
    torch.cuda.synchronize()
    for a, b, xa, xb in zip(views, dense, dXv, dXd):
        for k in ("W", "m", "v") + (("m_scale", "v_scale") if moment == "int8" else ()):
            assert torch.equal(a[k].view(torch.uint8), b[k].view(torch.uint8)), k
        assert torch.equal(xa, xb)
    assert (dXv[0].float().abs() > 0).any()


def test_store_g_matches_oracle_gradient():
    p = synth.make_problem("x", 300, 264, 520, seed=9)
    G = torch.empty(264, 520, device=DEV)
    fb.forge_wgrad_store_g(p.X.to(DEV), p.dY.to(DEV), G)
    Go, E = fo.wgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.X), with_abs=True)
    assert (np.abs(G.cpu().numpy().astype(np.float64) - Go) <= 300 * 2.0 ** -23 * E + 1e-30).all()


def test_result_independent_of_grid_size_and_repeatable():
    """Determinism (cf. identical digits across the paper's three variants): the
    result is bitwise independent of how many CTAs share the tile list."""
    p = synth.make_problem("x", 512, 1024, 1536, seed=11)
    outs = []
    d, _ = gpu_state(p, "fp32")
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 3, **HP)      # the product library
    torch.cuda.synchronize()
    outs.append(d)
    fb.use_profiling_library(True)          # FORGE_GRID exists only in the -DFORGE_PROFILING build
    try:
        for grid in (None, "1", "37", None):
            if grid:
                os.environ["FORGE_GRID"] = grid
            else:
                os.environ.pop("FORGE_GRID", None)
            d, _ = gpu_state(p, "fp32")
            fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 3, **HP)
            torch.cuda.synchronize()
            outs.append(d)
    finally:
        os.environ.pop("FORGE_GRID", None)
        fb.use_profiling_library(False)
    for d in outs[1:]:
        for k in ("W", "m", "v"):
            assert torch.equal(outs[0][k], d[k])


def test_randomised_shapes_strides_and_dispatch_paths_equal_the_twin_bitwise():
    """40 seeded random cases over T (1 ... 9000: ring, large-T ring, direct path), ragged out / in, the three moment dtypes,
    strided operand views: the fused call must equal store-G + the same update bit
    for bit.  (The gradient itself is checked against the oracle by the tests above.)"""
    import random
    rnd = random.Random(20260622)
    for it in range(40):
        moment = rnd.choice(["fp32", "bf16", "int8"])
        T = rnd.choice([1, 7, 33, 100, 512, 777, 2048, 4096, 8192, 8200]) if rnd.random() < 0.7 else rnd.randint(1, 3000)
        out = 8 * rnd.randint(1, 120)
        inn = 256 * rnd.randint(1, 4) if moment == "int8" else (16 * rnd.randint(1, 64) if moment == "bf16" or rnd.random() < 0.7 else 8 * rnd.randint(1, 128))
        if T >= 4096:
            out, inn = min(out, 520), min(inn, 768)
        p = synth.make_problem("f", T, out, inn, seed=5000 + it)
        d1, _ = gpu_state(p, moment)
        X, dY = d1["X"], d1["dY"]
        if rnd.random() < 0.4:                              # column slices of wider tensors: ldx / lddy
            wx = torch.zeros(T, inn + 24, dtype=torch.bfloat16, device=DEV)
            wy = torch.zeros(T, out + 40, dtype=torch.bfloat16, device=DEV)
            wx[:, 8:8 + inn], wy[:, 16:16 + out] = X, dY
            d1["X"], d1["dY"] = wx[:, 8:8 + inn], wy[:, 16:16 + out]
        d2 = {k: (v if k in ("X", "dY") else v.clone()) for k, v in d1.items()}
        fb.forge_wgrad_adamw_grouped([d1], *hp_args(5), {"fp32": fb.FP32, "bf16": fb.BF16, "int8": fb.INT8}[moment])
        G = torch.full((out, inn), float("nan"), device=DEV)
        fb.forge_wgrad_store_g(X, dY, G)
        fb.forge_adamw_from_g(G, d2["W"], d2["m"], d2["v"], 5, m_scale=d2.get("m_scale"), v_scale=d2.get("v_scale"), **HP)
        torch.cuda.synchronize()
        assert not torch.isnan(G).any()
        for k in d1:
            if k not in ("X", "dY"):
                assert torch.equal(d1[k].view(torch.uint8), d2[k].view(torch.uint8)), (it, moment, T, out, inn, k)


def test_stray_profiling_environment_cannot_change_a_product_result():
    """The ablation / grid / variant switches are compiled only into libforge_b200_prof.so: with the product library a
    FORGE_ABLATE=2 (\"no state loads / stores\") left over in the environment must change nothing."""
    ps = [synth.make_problem("a", 512, 640, 768, 21), synth.make_problem("b", 200, 136, 264, 22)]
    outs = []
    stray = {"FORGE_ABLATE": "2", "FORGE_GRID": "3", "FORGE_CFG": "7", "FORGE_POWER_STATE": "capped"}
    for env in ({}, stray):
        os.environ.update(env)
        try:
            devs = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in ps]
            fb.forge_wgrad_adamw_grouped(devs, *hp_args(4), fb.FP32)
            torch.cuda.synchronize()
        finally:
            for k in env:
                os.environ.pop(k, None)
        outs.append(devs)
    for a, b in zip(outs[0], outs[1]):
        for k in ("W", "m", "v"):
            assert torch.equal(a[k], b[k]), k
    assert not torch.equal(outs[0][0]["W"], ps[0].W.to(DEV))


def test_tuning_for_the_sustained_clock_is_bit_identical():
    """forge_set_tuning (include/forge.h): the instantiations for the boost and for the power-capped clock give the same
    bits, fp32 and bf16 moments, grouped launch, ragged shapes; an unknown value is rejected and changes nothing."""
    ps = [synth.make_problem("a", 512, 640, 768, 21), synth.make_problem("b", 200, 136, 264, 22), synth.make_problem("c", 512, 1024, 1536, 23)]
    for moment in ("fp32", "bf16"):
        outs, kernels = [], []
        for tuning in (fb.TUNE_BOOST_CLOCK, fb.TUNE_SUSTAINED_CLOCK):
            fb.forge_set_tuning(tuning)
            try:
                assert fb.forge_get_tuning() == tuning
                devs = [gpu_state(p, moment)[0] for p in ps]
                fb.forge_wgrad_adamw_grouped(devs, *hp_args(4), fb.FP32 if moment == "fp32" else fb.BF16)
                torch.cuda.synchronize()
                kernels.append(fb.lib().forge_last_kernel())
            finally:
                fb.forge_set_tuning(fb.TUNE_BOOST_CLOCK)
            outs.append(devs)
        assert kernels[0] != kernels[1]                    # two different instantiations did run
        for a, b in zip(outs[0], outs[1]):
            for k in ("W", "m", "v"):
                assert torch.equal(a[k], b[k]), (moment, k)
    assert fb.lib().forge_set_tuning(7) == 4 and fb.forge_get_tuning() == fb.TUNE_BOOST_CLOCK


def test_chunk_geometries_are_bit_identical():
    """Every instantiation sums the tokens in the same order and applies the same per-element update, so the chunk shape
    and ring depths are invisible in the results (FORGE_CFG, profiling build): grouped launch, ragged shapes."""
    ps = [synth.make_problem("a", 512, 640, 768, 21), synth.make_problem("b", 200, 136, 264, 22), synth.make_problem("c", 512, 1024, 1536, 23)]
    outs = []
    fb.use_profiling_library(True)
    try:
        for cfg in (None, "17", "5", "7"):
            if cfg:
                os.environ["FORGE_CFG"] = cfg
            else:
                os.environ.pop("FORGE_CFG", None)
            devs = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in ps]
            fb.forge_wgrad_adamw_grouped(devs, *hp_args(4), fb.FP32)
            torch.cuda.synchronize()
            outs.append(devs)
    finally:
        os.environ.pop("FORGE_CFG", None)
        fb.use_profiling_library(False)
    for devs in outs[1:]:
        for a, b in zip(outs[0], devs):
            for k in ("W", "m", "v"):
                assert torch.equal(a[k], b[k]), k
    assert not torch.equal(outs[0][0]["W"], ps[0].W.to(DEV))


def test_grouped_call_is_cuda_graph_capturable_and_replays_bitwise():
    """The ABI enqueues on the caller's stream, allocates nothing and synchronises nothing, so a layer's call (and the
    layer-backward call: dgrad launch + fused launch) can be captured into a CUDA graph and replayed: the replay applies
    the same step to whatever the buffers hold, bit-identical to the eager call on the same state."""
    ps = [synth.make_problem("a", 512, 640, 768, 41), synth.make_problem("b", 200, 136, 264, 42)]
    eager = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in ps]
    graph = [dict(X=d["X"], dY=d["dY"], W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p, d in zip(ps, eager)]
    dX_e = [torch.zeros(p.T, p.inn, dtype=torch.bfloat16, device=DEV) for p in ps]
    dX_g = [torch.zeros(p.T, p.inn, dtype=torch.bfloat16, device=DEV) for p in ps]
    fb.forge_layer_backward_grouped(eager, dX_e, *hp_args(6), fb.FP32)           # warm-up: function attributes are set
    for d, p in zip(eager, ps):
        d["W"].copy_(p.W.to(DEV)); d["m"].copy_(p.m.to(DEV)); d["v"].copy_(p.v.to(DEV))
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        g.capture_begin()
        fb.forge_layer_backward_grouped(graph, dX_g, *hp_args(6), fb.FP32, stream=side)
        g.capture_end()
    torch.cuda.synchronize()
    for d, p in zip(graph, ps):
        assert torch.equal(d["W"], p.W.to(DEV))                                   # capture did not execute anything
    for _ in range(2):                                                             # two replays = two eager calls
        g.replay()
        fb.forge_layer_backward_grouped(eager, dX_e, *hp_args(6), fb.FP32)
    torch.cuda.synchronize()
    for a, b, x, y in zip(eager, graph, dX_e, dX_g):
        for k in ("W", "m", "v"):
            assert torch.equal(a[k], b[k]), k
        assert torch.equal(x, y)
    assert not torch.equal(graph[0]["W"], ps[0].W.to(DEV))


# ------------------------------------------------------------------------------ properties ---
def test_lr_zero_keeps_w_and_inputs_untouched_moments_move():
    p = synth.make_problem("x", 256, 256, 512, seed=13)
    d, _ = gpu_state(p, "fp32")
    X0, dY0, W0, m0 = d["X"].clone(), d["dY"].clone(), d["W"].clone(), d["m"].clone()
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 4, 0.0, HP["beta1"], HP["beta2"], HP["eps"], HP["wd"])
    torch.cuda.synchronize()
    assert torch.equal(d["W"], W0) and torch.equal(d["X"], X0) and torch.equal(d["dY"], dY0)
    assert not torch.equal(d["m"], m0)


def test_grouped_more_than_eight_problems_and_no_workspace():
    probs = [synth.make_problem(f"p{i}", 64, 128, 256, seed=200 + i) for i in range(11)]
    ds, os_ = zip(*[gpu_state(p, "fp32") for p in probs])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    before = fb.forge_launch_count()
    fb.forge_wgrad_adamw_grouped(list(ds), 2, *pu.hp_tuple(HP), 0)
    torch.cuda.synchronize()
    assert fb.forge_launch_count() - before == 2               # 8 + 3
    assert torch.cuda.mem_get_info()[0] == free0               # the library allocated nothing: no dW
    for p, d, o in zip(probs, ds, os_):
        G, E = fo.wgrad(o["dY"], o["X"], with_abs=True)
        W_prev = o["W"].copy()
        fo.adamw_fp32(o["W"], o["m"], o["v"], G, 2, *pu.hp_tuple(HP))
        tol = pu.Tol(G.shape)
        e = tol.step(G, E, 64, HP)
        pu.check_fp(pu.to_np(d["W"]), pu.to_np(d["m"]), pu.to_np(d["v"]), o["W"], o["m"], o["v"], G, e, tol, HP, W_prev=W_prev)


def test_bad_arguments_leave_state_untouched_on_gpu():
    p = synth.make_problem("x", 64, 128, 256, seed=17)
    d, _ = gpu_state(p, "fp32")
    W0, m0 = d["W"].clone(), d["m"].clone()
    st = fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 0, check=False, **HP)
    assert st == 4
    with pytest.raises(fb.ForgeError):
        fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"][:, 1:], d["v"], 1, **HP)   # misaligned
    torch.cuda.synchronize()
    assert torch.equal(d["W"], W0) and torch.equal(d["m"], m0)


def test_host_buffer_entry_point_matches_device_path():
    p = synth.make_problem("x", 128, 256, 512, seed=19)
    d, _ = gpu_state(p, "fp32")
    fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], 6, **HP)
    h = dict(X=p.X.clone().pin_memory(), dY=p.dY.clone().pin_memory(), W=p.W.clone().pin_memory(),
             m=p.m.clone().pin_memory(), v=p.v.clone().pin_memory())
    fb.forge_wgrad_adamw_host(h["X"], h["dY"], h["W"], h["m"], h["v"], 6, **HP)
    torch.cuda.synchronize()
    for k in ("W", "m", "v"):
        assert torch.equal(d[k].cpu(), h[k])


def test_config4_full_stack_reverse_order_sampled_rows():
    """BASELINE.json configs[4] at full size: 32 layers + lm_head resident (75 GB), one step in reverse
    layer order through the grouped entry; lm_head and three layers are checked on sampled rows against
    the oracle (rows are independent, so a row subset is an exact oracle for those rows)."""
    from paper_2606_22932_b200 import stack
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.skip("needs ~80 GB of free device memory")
    dev = torch.device("cuda:0")
    st = stack.build_stack(dev, tokens=512)
    assert st.params == 32 * 218103808 + 128256 * 4096 and len(st.layers) == 33
    hp = synth.HP_DEFAULT
    picks = [(32, 0), (31, 6), (16, 4), (0, 0), (0, 1)]          # lm_head, L31.down, L16.gate, L0.q, L0.k
    before = {}
    for li, pi in picks:
        d = st.layers[li][pi]
        out = d["W"].shape[0]
        rows = pu.spread_rows(out, 16, 128) if li == 32 else pu.sample_rows(out, seed=li)   # lm_head: 1/16 of its rows
        before[(li, pi)] = [(r0, r1, synth.bf16_bits(d["W"][r0:r1]).copy(), d["m"][r0:r1].cpu().numpy().copy(),
                             d["v"][r0:r1].cpu().numpy().copy()) for r0, r1 in rows]
    torch.cuda.reset_peak_memory_stats()
    base_alloc = torch.cuda.memory_allocated()
    n = stack.step_fused(st, 10, hp)
    torch.cuda.synchronize()
    assert n == 33                                               # one launch per layer + lm_head
    assert torch.cuda.max_memory_allocated() == base_alloc       # nothing gradient-shaped was allocated
    for li, pi in picks:
        d = st.layers[li][pi]
        dYb, Xb = synth.bf16_bits(d["dY"]), synth.bf16_bits(d["X"])
        T = d["X"].shape[0]
        for r0, r1, Wb, m0, v0 in before[(li, pi)]:
            G, E = fo.wgrad(dYb, Xb, rows=(r0, r1), with_abs=True)
            Wp = Wb.copy()
            tol = pu.Tol(G.shape)
            e = tol.step(G, E, T, hp)
            wprop = pu.w_propagated("fp32", Wb, m0, v0, G, e, 10, hp)
            fo.adamw_fp32(Wb, m0, v0, G, 10, *pu.hp_tuple(hp))
            pu.check_fp(synth.bf16_bits(d["W"][r0:r1]), d["m"][r0:r1].cpu().numpy(), d["v"][r0:r1].cpu().numpy(),
                                 Wb, m0, v0, G, e, tol, hp, label=f"{d['name']}[{r0}:{r1}]", W_prev=Wp, w_prop=wprop)


def test_layer_backward_dgrad_reads_pre_update_weights_then_fused_step():
    """SURVEY.md 8(f) rank 2 (Alg. 1 line 1; 64; 296): forge_layer_backward_grouped computes
    dX = dY . W from the PRE-update W, then the fused step; W/m/v must equal the plain grouped call bit for bit."""
    ps = [synth.make_problem("a", 200, 136, 264, 31), synth.make_problem("b", 96, 256, 512, 32)]
    probs, twins, dXs = [], [], []
    for p in ps:
        probs.append(dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()))
        twins.append(dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()))
        dXs.append(torch.full((p.T, p.inn), float("nan"), dtype=torch.bfloat16, device=DEV))
    fb.forge_layer_backward_grouped(probs, dXs, *hp_args(10), fb.FP32)
    fb.forge_wgrad_adamw_grouped(twins, *hp_args(10), fb.FP32)
    torch.cuda.synchronize()
    for p, d, t, dX in zip(ps, probs, twins, dXs):
        assert torch.equal(d["W"], t["W"]) and torch.equal(d["m"], t["m"]) and torch.equal(d["v"], t["v"])
        assert not torch.equal(d["W"].cpu(), p.W)                                    # the step did happen
        ref = fo.dgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.W))                  # oracle, PRE-update W
        got = fo.bf16_to_f64(synth.bf16_bits(dX))
        bound = p.out * 2.0 ** -23 * (np.abs(fo.bf16_to_f64(synth.bf16_bits(p.dY))) @ np.abs(fo.bf16_to_f64(synth.bf16_bits(p.W))))
        assert np.all(np.abs(got - ref) <= pu.bf16_ulp(ref) + bound), np.abs(got - ref).max()
        assert float((synth.bf16_bits(dX) == fo.f64_to_bf16(ref)).mean()) > 0.98
        post = fo.dgrad(synth.bf16_bits(p.dY), synth.bf16_bits(d["W"]))              # what a mis-ordered call would give
        assert float((synth.bf16_bits(dX) == fo.f64_to_bf16(post)).mean()) < 0.9
    # a bad argument in the second problem: nothing is enqueued, nothing changes
    W0 = probs[0]["W"].clone()
    bad = [probs[0], dict(probs[1], m=None)]
    assert fb.forge_layer_backward_grouped(bad, dXs, *hp_args(11), fb.FP32, check=False) == 1
    torch.cuda.synchronize()
    assert torch.equal(probs[0]["W"], W0)


def test_dgrad_kernel_multi_tile_grouped_depths_and_strided_dy():
    """The hand-written tcgen05 dgrad (csrc/dgrad_kernel.cuh) against the oracle's plain definition
    dX[t,q] = sum_p dY[t,p] W[p,q] (Alg. 1 line 1) on a group whose tiles differ in depth (the
    longest-first assignment), span several 256 x 256 tiles with ragged T / in / out tails, and read dY as a column
    slice of a wider tensor (lddy)."""
    shapes = [("a", 512, 1024, 768), ("b", 300, 2056, 520), ("c", 700, 136, 264), ("d", 128, 4096, 256), ("e", 1, 64, 8)]
    ps = [synth.make_problem(n, T, o, i, 70 + k) for k, (n, T, o, i) in enumerate(shapes)]
    probs, dXs = [], []
    for k, p in enumerate(ps):
        dY = p.dY.to(DEV)
        if k % 2 == 1:                                   # strided view
            wide = torch.zeros(p.T, p.out + 48, dtype=torch.bfloat16, device=DEV)
            wide[:, 24:24 + p.out] = dY
            dY = wide[:, 24:24 + p.out]
        probs.append(dict(X=p.X.to(DEV), dY=dY, W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()))
        dXs.append(torch.full((p.T, p.inn), float("nan"), dtype=torch.bfloat16, device=DEV))
    launches0 = fb.forge_launch_count()
    fb.forge_layer_backward_grouped(probs, dXs, *hp_args(10), fb.FP32)
    torch.cuda.synchronize()
    assert fb.forge_launch_count() - launches0 == 2          # one dgrad launch + one fused launch
    for p, dX in zip(ps, dXs):
        dYf, Wf = fo.bf16_to_f64(synth.bf16_bits(p.dY)), fo.bf16_to_f64(synth.bf16_bits(p.W))
        ref = fo.dgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.W))
        got = fo.bf16_to_f64(synth.bf16_bits(dX))
        assert not np.isnan(got).any()
        bound = p.out * 2.0 ** -23 * (np.abs(dYf) @ np.abs(Wf))
        assert np.all(np.abs(got - ref) <= pu.bf16_ulp(ref) + bound), (p.name, np.abs(got - ref).max())
        assert float((synth.bf16_bits(dX) == fo.f64_to_bf16(ref)).mean()) > 0.98, p.name


def test_grouped_host_entry_matches_device_path_bitwise():
    """forge_wgrad_adamw_grouped_host (pipelined H2D / step / D2H): same bits as the device-resident grouped call."""
    ps = [synth.make_problem("a", 200, 136, 264, 61), synth.make_problem("b", 96, 256, 512, 62), synth.make_problem("c", 64, 128, 256, 63)]
    host = [dict(X=p.X.pin_memory(), dY=p.dY.pin_memory(), W=p.W.clone().pin_memory(), m=p.m.clone().pin_memory(),
                 v=p.v.clone().pin_memory()) for p in ps]
    devs = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in ps]
    fb.forge_wgrad_adamw_grouped_host(host, *hp_args(10), fb.FP32)
    fb.forge_wgrad_adamw_grouped(devs, *hp_args(10), fb.FP32)
    torch.cuda.synchronize()
    for h, d, p in zip(host, devs, ps):
        assert torch.equal(h["W"], d["W"].cpu()) and torch.equal(h["m"], d["m"].cpu()) and torch.equal(h["v"], d["v"].cpu())
        assert not torch.equal(h["W"], p.W)

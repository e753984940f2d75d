"""GPU parity for the other coordinate-wise optimizer families:
forge_wgrad_step_grouped through the C ABI against oracle/forge_oracle_families.c on the same seeded inputs.
Tolerance: W within 1 bf16 ulp of the oracle (+ the fp32 evaluation error of the update) wherever the
gradient is determined (|g| > 4e, e the fp32 accumulation bound of north_star), elsewhere within the
family's largest step; state to relative 1e-4 plus the propagated accumulation error."""
import numpy as np
import pytest
import torch

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import binding as fb
from paper_2606_22932_b200 import synth
import parity_util as pu

pytestmark = pytest.mark.gpu
DEV = "cuda"
F = np.float32

CASES = {
    "sgd": dict(lr=1e-2, wd=0.05),
    "momentum": dict(lr=1e-2, wd=0.05, momentum=0.9),
    "nesterov": dict(lr=1e-2, wd=0.05, momentum=0.8, nesterov=True),
    "lion": dict(lr=1e-4, beta1=0.9, beta2=0.99, wd=0.1),
    "rmsprop": dict(lr=1e-3, beta2=0.99, eps=1e-8, wd=0.01),
    "adagrad": dict(lr=1e-2, eps=1e-10, wd=0.0),
    "adamax": dict(lr=2e-3, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.01),
    "nadam": dict(lr=2e-3, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.01),
    "radam": dict(lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.01),
}


def run_case(name, T, out, inn, steps, state_bf16=False, seed=3):
    fam = "momentum" if name == "nesterov" else name
    kw = dict(beta1=0.9, beta2=0.999, eps=1e-8, wd=0.0, momentum=0.0, nesterov=False)
    kw.update(CASES[name])
    lr = kw.pop("lr")
    ns = fb.FAMILY_STATES[fam]
    p0 = synth.make_problem("f", T, out, inn, seed, sigma_dy=1e-2)
    Wg = p0.W.to(DEV).clone()
    Wo = synth.bf16_bits(p0.W).copy()
    sdt = torch.bfloat16 if state_bf16 else torch.float32
    # non-trivial initial state (v-like states non-negative), identical bits on both sides
    init = [p0.m * 10, p0.v.sqrt() if fam == "adamax" else p0.v * 100][:ns] if fam not in ("rmsprop", "adagrad") else [p0.v * 100]
    sg = [t.to(sdt).to(DEV) for t in init]
    so = [synth.bf16_bits(t.to(sdt)).copy() if state_bf16 else t.numpy().copy() for t in init]
    exact = []
    for step in steps:
        pin = synth.make_problem("f", T, out, inn, seed + step, sigma_dy=1e-2)
        X, dY = pin.X.to(DEV), pin.dY.to(DEV)
        prob = dict(X=X, dY=dY, W=Wg, m=sg[0] if ns >= 1 else None, v=sg[1] if ns >= 2 else None)
        fb.forge_wgrad_step_grouped([prob], fam, step, lr, state_dtype=fb.BF16 if state_bf16 else fb.FP32, **kw)
        G, E = fo.wgrad(synth.bf16_bits(pin.dY), synth.bf16_bits(pin.X), with_abs=True)
        Wprev = fo.bf16_to_f64(Wo)
        fo.family_step(fam, Wo, *(so + [None] * (2 - ns)), G, step, lr, kw["beta1"], kw["beta2"], kw["eps"], kw["wd"],
                       kw["momentum"], kw["nesterov"])
        torch.cuda.synchronize()
        Wr, Wd = fo.bf16_to_f64(Wo), fo.bf16_to_f64(synth.bf16_bits(Wg))
        e = T * 2.0 ** -23 * E
        dW = np.abs(Wd - Wr)
        # one bf16 ulp (the larger binade's when the two results straddle a power of two) + fp32 evaluation error
        # and, for the rules that are LINEAR in g (SGD, momentum), the accumulation bound itself: dW = lr * dg
        # (it only matters where W - lr*g cancels to ~0 and an ulp of the result is far below fp32 eps of W)
        ulp = (np.maximum(pu.bf16_ulp(Wr), pu.bf16_ulp(Wd)) + 2.0 ** -20 * (np.abs(Wprev) + np.abs(Wr - Wprev))
               + 2 * lr * e)
        big = max(4 * lr, 4 * np.abs(Wr - Wprev).max())            # the family's largest step (sign-like rules flip by 2 steps)
        sure = np.abs(G) > 4 * e
        bad = np.where(sure, dW > len(exact) * ulp + ulp, dW > big)
        assert not bad.any(), f"{name} step {step}: {bad.sum()} W outside tolerance, worst {dW.max():.3e}"
        exact.append(float((synth.bf16_bits(Wg) == Wo).mean()))
        for a, b in zip(sg, so):
            ag = fo.bf16_to_f64(synth.bf16_bits(a)) if state_bf16 else a.cpu().numpy().astype(np.float64)
            bo = fo.bf16_to_f64(b) if state_bf16 else b.astype(np.float64)
            tol = (2.0 ** -7 if state_bf16 else 2e-4) * np.abs(bo) + 8 * e * (1 + 2 * np.abs(G)) + 1e-30
            assert np.all(np.abs(ag - bo) <= tol), f"{name} step {step}: state off by {np.abs(ag - bo).max():.3e}"
        # chain both sides from the ORACLE's values so one-ulp flips do not accumulate into the next step's check
        Wg.copy_(synth.bits_to_bf16(Wo).to(DEV))
        for a, b in zip(sg, so):
            a.copy_((synth.bits_to_bf16(b) if state_bf16 else torch.from_numpy(b)).to(DEV))
    assert min(exact) > 0.98, f"{name}: only {min(exact):.4f} of W bit-identical to the oracle"


@pytest.mark.parametrize("name", list(CASES))
def test_family_small_shapes_three_steps_fp32_state(name):
    run_case(name, T=200, out=136, inn=264, steps=(1, 2, 7))


@pytest.mark.parametrize("name", ["momentum", "lion", "rmsprop", "adamax", "radam"])
def test_family_bf16_state(name):
    run_case(name, T=96, out=256, inn=512, steps=(1, 6), state_bf16=True)


@pytest.mark.parametrize("name", ["sgd", "lion", "nadam"])
def test_family_large_t_variant(name):
    run_case(name, T=2048, out=256, inn=512, steps=(3,))


def test_family_argument_validation():
    p = synth.make_problem("f", 64, 128, 256, 1)
    X, dY, W, m = p.X.to(DEV), p.dY.to(DEV), p.W.to(DEV), p.m.to(DEV)
    W0 = W.clone()
    # SGD must not be given state; momentum must; int8 state is AdamW-only; bad momentum
    assert fb.forge_wgrad_step_grouped([dict(X=X, dY=dY, W=W, m=m, v=None)], "sgd", 1, 1e-2, check=False) == 1
    assert fb.forge_wgrad_step_grouped([dict(X=X, dY=dY, W=W, m=None, v=None)], "momentum", 1, 1e-2, check=False) == 1
    assert fb.forge_wgrad_step_grouped([dict(X=X, dY=dY, W=W, m=m, v=None)], "lion", 1, 1e-2, state_dtype=fb.INT8, check=False) == 5
    assert fb.forge_wgrad_step_grouped([dict(X=X, dY=dY, W=W, m=m, v=None)], "momentum", 1, 1e-2, momentum=1.5, check=False) == 4
    torch.cuda.synchronize()
    assert torch.equal(W, W0)


@pytest.mark.parametrize("T,out,inn,bf16", [(200, 136, 264, False), (512, 384, 768, True), (2048, 256, 512, False)])
def test_accumulate_into_state_matches_oracle(T, out, inn, bf16):
    """B <- mu*B + dY^T X with no weight and no gradient buffer.
    |dB| <= e (the fp32 accumulation bound of north_star) + the storage rounding."""
    mu = 0.95
    p = synth.make_problem("a", T, out, inn, 17, sigma_dy=1e-2)
    B0 = p.m * 100
    sdt = torch.bfloat16 if bf16 else torch.float32
    Bg = B0.to(sdt).to(DEV)
    Bo = synth.bf16_bits(B0.to(sdt)).copy() if bf16 else B0.numpy().copy()
    X, dY = p.X.to(DEV), p.dY.to(DEV)
    X0, dY0 = X.clone(), dY.clone()
    n0 = fb.forge_launch_count()
    fb.forge_wgrad_accumulate_grouped([dict(X=X, dY=dY, W=None, m=Bg, v=None)], mu, state_dtype=fb.BF16 if bf16 else fb.FP32)
    torch.cuda.synchronize()
    assert fb.forge_launch_count() - n0 == 1 and torch.equal(X, X0) and torch.equal(dY, dY0)
    G, E = fo.wgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.X), with_abs=True)
    fo.accumulate(Bo, G, mu)
    e = T * 2.0 ** -23 * E
    got = fo.bf16_to_f64(synth.bf16_bits(Bg)) if bf16 else Bg.cpu().numpy().astype(np.float64)
    ref = fo.bf16_to_f64(Bo) if bf16 else Bo.astype(np.float64)
    tol = e + (2.0 ** -7 if bf16 else 2.0 ** -22) * np.abs(ref)
    assert np.all(np.abs(got - ref) <= tol), np.abs(got - ref).max()
    # the worst-case bound must not hide a systematic error: bf16 results are almost all bit-identical, fp32 ones
    # agree to the typical (not worst-case) fp32 accumulation error
    same = (synth.bf16_bits(Bg) == Bo).mean() if bf16 else np.isclose(got, ref, rtol=2e-5, atol=1e-9).mean()
    assert same > 0.97
    # W / v must be absent: the call refuses and touches nothing
    assert fb.forge_wgrad_accumulate_grouped([dict(X=X, dY=dY, W=p.W.to(DEV), m=Bg, v=None)], mu, check=False) == 5


def test_adamw_stochastic_rounding_store_matches_oracle_generator():
    """the SR store.  Both sides implement the same counter-based
    generator, so the result is deterministic: m, v as the RNE call; W one of the two bf16 neighbours of W', equal
    to the oracle's choice except where the kernel's fp32 W' and fp32(oracle W') differ in their low bits."""
    ps = [synth.make_problem("a", 200, 136, 264, 41), synth.make_problem("b", 96, 256, 512, 42)]
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    probs = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in ps]
    twins = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in ps]
    again = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone()) for p in ps]
    seed = (7 << 40) + 12345
    fb.forge_wgrad_adamw_sr_grouped(probs, 10, *hpt, fb.FP32, seed)
    fb.forge_wgrad_adamw_sr_grouped(again, 10, *hpt, fb.FP32, seed)
    fb.forge_wgrad_adamw_grouped(twins, 10, *hpt, fb.FP32)
    torch.cuda.synchronize()
    for i, (p, d, t, a) in enumerate(zip(ps, probs, twins, again)):
        assert torch.equal(d["m"], t["m"]) and torch.equal(d["v"], t["v"])           # only the store of W differs
        assert torch.equal(d["W"], a["W"])                                           # reproducible for a fixed seed
        Wo, mo, vo = synth.bf16_bits(p.W).copy(), p.m.numpy().copy(), p.v.numpy().copy()
        G = fo.wgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.X))
        fo.adamw_fp32_sr(Wo, mo, vo, G, 10, *hpt, seed=seed, stream=i)
        Wg = synth.bf16_bits(d["W"])
        assert np.abs(Wg.astype(np.int32) - Wo.astype(np.int32)).max() <= 1          # always a neighbour
        assert float((Wg == Wo).mean()) > 0.995, float((Wg == Wo).mean())
        Wr = synth.bf16_bits(t["W"])
        assert np.abs(Wg.astype(np.int32) - Wr.astype(np.int32)).max() <= 1 and float((Wg != Wr).mean()) > 0.2
    # bf16 moments run too; int8 is refused
    fb.forge_wgrad_adamw_sr_grouped([dict(X=ps[0].X.to(DEV), dY=ps[0].dY.to(DEV), W=ps[0].W.to(DEV).clone(),
                                          m=ps[0].m.to(torch.bfloat16).to(DEV), v=ps[0].v.to(torch.bfloat16).to(DEV))],
                                    3, *hpt, fb.BF16, 5)
    assert fb.forge_wgrad_adamw_sr_grouped(probs, 11, *hpt, fb.INT8, seed, check=False) == 5
    torch.cuda.synchronize()


@pytest.mark.parametrize("T,out,inn", [(200, 136, 272), (512, 384, 768), (2048, 256, 512)])
def test_adamw_fp8_moments_delayed_scaling(T, out, inn):
    """SURVEY.md 8(f) rank 1 (reading S17): e4m3 moments, one scale per tensor,
    delayed scaling.  Codes within one e4m3 step of the oracle's (the decision x*inv -> e4m3 is taken in fp32 on
    both sides; they differ only where the fp32 m', v' differ), W as for fp32 moments, the reported amax to 1e-5."""
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    p = synth.make_problem("f8", T, out, inn, 51)
    mq, ms = fo.fp8_quantize(p.m.numpy())
    vq, vs = fo.fp8_quantize(p.v.numpy())
    Wg = p.W.to(DEV).clone()
    mg, vg = torch.from_numpy(mq.copy()).to(DEV), torch.from_numpy(vq.copy()).to(DEV)
    msg, vsg = torch.from_numpy(ms.copy()).to(DEV), torch.from_numpy(vs.copy()).to(DEV)
    fb.forge_wgrad_adamw(p.X.to(DEV), p.dY.to(DEV), Wg, mg, vg, 10, *hpt, m_scale=msg, v_scale=vsg, moment_dtype=fb.FP8)
    torch.cuda.synchronize()
    Wo, mo, vo, mso, vso = synth.bf16_bits(p.W).copy(), mq.copy(), vq.copy(), ms.copy(), vs.copy()
    G, E = fo.wgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.X), with_abs=True)
    Wprev = fo.bf16_to_f64(Wo)
    fo.adamw_fp8(Wo, mo, vo, mso, vso, G, 10, *hpt)
    e = T * 2.0 ** -23 * E
    # W: the fp32-moment criterion of north_star
    Wr, Wd = fo.bf16_to_f64(Wo), fo.bf16_to_f64(synth.bf16_bits(Wg))
    ulp = np.maximum(pu.bf16_ulp(Wr), pu.bf16_ulp(Wd)) + 2.0 ** -20 * (np.abs(Wprev) + np.abs(Wr - Wprev))
    bad = np.where(np.abs(G) > 4 * e, np.abs(Wd - Wr) > ulp, np.abs(Wd - Wr) > 2 * hp["lr"] + ulp)
    assert not bad.any() and float((synth.bf16_bits(Wg) == Wo).mean()) > 0.99
    # codes: same sign, magnitude code within 1 (adjacent e4m3 values), almost all identical
    for got, ref in ((mg.cpu().numpy(), mo), (vg.cpu().numpy(), vo)):
        dm = np.abs((got & 0x7F).astype(int) - (ref & 0x7F).astype(int))
        assert dm.max() <= 1 and float((got == ref).mean()) > 0.99
        assert np.all(((got ^ ref) & 0x80 == 0) | ((got & 0x7F) <= 1) & ((ref & 0x7F) <= 1))
    # scale in use untouched, amax of this step reported for the next step's scale
    msn, vsn = msg.cpu().numpy(), vsg.cpu().numpy()
    assert msn[0] == ms[0] and vsn[0] == vs[0]
    assert np.isclose(msn[1], mso[1], rtol=1e-4) and np.isclose(vsn[1], vso[1], rtol=1e-4)
    # missing scales are refused
    assert fb.forge_wgrad_adamw(p.X.to(DEV), p.dY.to(DEV), Wg, mg, vg, 11, *hpt, moment_dtype=fb.FP8, check=False) == 1


# ------------------------------------------------------------------ full layer size, sampled rows
@pytest.fixture(scope="module")
def layer_cpu():
    return synth.make_layer(512, seed=synth.BASE_SEED + 1)


@pytest.mark.parametrize("family,every_row", [("momentum", True), ("lion", False), ("sgd", False)])
def test_full_layer_family_grouped_sampled_rows(layer_cpu, family, every_row):
    """The 7 projections of a Llama-3.1-8B layer at full size in ONE grouped launch (the configuration
    `bench.py --optimizer` times); the oracle is exact on a deterministic sample of rows (rows are independent) --
    for SGD with momentum on EVERY row of the layer."""
    kw = dict(beta1=0.9, beta2=0.99, eps=1e-8, wd=0.05, momentum=0.9, nesterov=False)
    lr = 1e-4 if family == "lion" else 1e-2
    ns = fb.FAMILY_STATES[family]
    devs = [dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=(p.m * 10).to(DEV) if ns else None, v=None)
            for p in layer_cpu]
    n0 = fb.forge_launch_count()
    fb.forge_wgrad_step_grouped(devs, family, 4, lr, **kw)
    torch.cuda.synchronize()
    assert fb.forge_launch_count() - n0 == 1
    for p, d in zip(layer_cpu, devs):
        dYb, Xb = synth.bf16_bits(p.dY), synth.bf16_bits(p.X)
        ranges = [(r0, min(p.out, r0 + 512)) for r0 in range(0, p.out, 512)] if every_row else pu.sample_rows(p.out)
        for r0, r1 in ranges:
            G, E = fo.wgrad(dYb, Xb, rows=(r0, r1), with_abs=True)
            Wo = synth.bf16_bits(p.W[r0:r1]).copy()
            Wprev = fo.bf16_to_f64(Wo)
            so = [(p.m[r0:r1] * 10).numpy().copy()] if ns else []
            m_before = so[0].astype(np.float64) if ns else None
            fo.family_step(family, Wo, *(so + [None] * (2 - ns)), G, 4, lr, kw["beta1"], kw["beta2"], kw["eps"], kw["wd"],
                           kw["momentum"], kw["nesterov"])
            e = 512 * 2.0 ** -23 * E
            Wr, Wd = fo.bf16_to_f64(Wo), fo.bf16_to_f64(synth.bf16_bits(d["W"][r0:r1]))
            ulp = (np.maximum(pu.bf16_ulp(Wr), pu.bf16_ulp(Wd)) + 2.0 ** -20 * (np.abs(Wprev) + np.abs(Wr - Wprev)) + 2 * lr * e)
            sure = np.abs(G) > 4 * e if family != "lion" else np.abs(0.9 * m_before + 0.1 * G) > 4 * e   # Lion: the sign of c
            bad = np.where(sure, np.abs(Wd - Wr) > ulp, np.abs(Wd - Wr) > 4 * lr + ulp)
            assert not bad.any(), f"{family} {p.name}[{r0}:{r1}]: {bad.sum()} W outside tolerance"
            assert float((synth.bf16_bits(d["W"][r0:r1]) == Wo).mean()) > 0.98
            if ns:
                got = d["m"][r0:r1].cpu().numpy().astype(np.float64)
                assert np.all(np.abs(got - so[0]) <= 2e-4 * np.abs(so[0]) + 4 * e)


def test_full_layer_fp8_grouped_sampled_rows(layer_cpu):
    """fp8 moments at full cfg-1 size, one grouped launch; codes / W / amax against the oracle on sampled rows."""
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    devs, keep = [], []
    for p in layer_cpu:
        mq, ms = fo.fp8_quantize(p.m.numpy())
        vq, vs = fo.fp8_quantize(p.v.numpy())
        keep.append((mq, ms, vq, vs))
        devs.append(dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=torch.from_numpy(mq.copy()).to(DEV),
                         v=torch.from_numpy(vq.copy()).to(DEV), m_scale=torch.from_numpy(ms.copy()).to(DEV),
                         v_scale=torch.from_numpy(vs.copy()).to(DEV)))
    n0 = fb.forge_launch_count()
    fb.forge_wgrad_adamw_grouped(devs, 10, *hpt, fb.FP8)
    torch.cuda.synchronize()
    assert fb.forge_launch_count() - n0 == 1
    for p, d, (mq, ms, vq, vs) in zip(layer_cpu, devs, keep):
        dYb, Xb = synth.bf16_bits(p.dY), synth.bf16_bits(p.X)
        amax_rows = 0.0
        for r0, r1 in pu.sample_rows(p.out):
            G = fo.wgrad(dYb, Xb, rows=(r0, r1))
            Wo, mo, vo, mso, vso = synth.bf16_bits(p.W[r0:r1]).copy(), mq[r0:r1].copy(), vq[r0:r1].copy(), ms.copy(), vs.copy()
            fo.adamw_fp8(Wo, mo, vo, mso, vso, G, 10, *hpt)
            amax_rows = max(amax_rows, float(mso[1]))
            assert float((synth.bf16_bits(d["W"][r0:r1]) == Wo).mean()) > 0.99
            for got, ref in ((d["m"][r0:r1].cpu().numpy(), mo), (d["v"][r0:r1].cpu().numpy(), vo)):
                assert np.abs((got & 0x7F).astype(int) - (ref & 0x7F).astype(int)).max() <= 1
                assert float((got == ref).mean()) > 0.99
        got_amax = float(d["m_scale"].cpu()[1])
        assert got_amax >= amax_rows * (1 - 1e-5)                  # the tensor-wide amax covers every sampled row
        assert float(d["m_scale"].cpu()[0]) == float(ms[0])


@pytest.mark.parametrize("T,out,inn", [(1, 8, 16), (33, 8, 16), (7, 136, 24)])
def test_tiny_and_ragged_shapes_new_entries(T, out, inn):
    """Degenerate sizes through the widened entry points: one token, one 8-row strip, ragged everything."""
    p = synth.make_problem("t", T, out, inn, 71, sigma_dy=1e-2)
    G = fo.wgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.X))
    X, dY = p.X.to(DEV), p.dY.to(DEV)
    # momentum
    W, m = p.W.to(DEV).clone(), (p.m * 10).to(DEV)
    fb.forge_wgrad_step_grouped([dict(X=X, dY=dY, W=W, m=m, v=None)], "momentum", 2, 1e-2, momentum=0.9)
    Wo, mo = synth.bf16_bits(p.W).copy(), (p.m * 10).numpy().copy()
    fo.family_step("momentum", Wo, mo, None, G, 2, 1e-2, momentum=0.9)
    torch.cuda.synchronize()
    assert np.abs(synth.bf16_bits(W).astype(int) - Wo.astype(int)).max() <= 1
    assert np.allclose(m.cpu().numpy(), mo, rtol=1e-5, atol=1e-9)
    # accumulate
    B = (p.m * 100).to(DEV)
    fb.forge_wgrad_accumulate_grouped([dict(X=X, dY=dY, W=None, m=B, v=None)], 0.5)
    Bo = (p.m * 100).numpy().copy()
    fo.accumulate(Bo, G, 0.5)
    torch.cuda.synchronize()
    assert np.allclose(B.cpu().numpy(), Bo, rtol=1e-5, atol=1e-9)
    # SR store: always a neighbour of the RNE result
    Ws, ms_, vs_ = p.W.to(DEV).clone(), p.m.to(DEV).clone(), p.v.to(DEV).clone()
    Wr, mr, vr = p.W.to(DEV).clone(), p.m.to(DEV).clone(), p.v.to(DEV).clone()
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    fb.forge_wgrad_adamw_sr_grouped([dict(X=X, dY=dY, W=Ws, m=ms_, v=vs_)], 3, *hpt, fb.FP32, 77)
    fb.forge_wgrad_adamw_grouped([dict(X=X, dY=dY, W=Wr, m=mr, v=vr)], 3, *hpt, fb.FP32)
    torch.cuda.synchronize()
    assert np.abs(synth.bf16_bits(Ws).astype(int) - synth.bf16_bits(Wr).astype(int)).max() <= 1 and torch.equal(ms_, mr)


@pytest.mark.parametrize("mode", ["fp32", "bf16", "int8", "fp8", "sr", "momentum", "sgd", "accum"])
def test_every_mode_is_bitwise_repeatable_on_a_ragged_group(mode):
    """Race evidence without a sanitizer (compute-sanitizer is closed on this pool): every entry point, on a group of
    ragged problems spanning many tiles and both T regimes, gives bit-identical results on 8 repeated runs from the
    same state (a missed barrier or an early slot reuse would show up as run-to-run differences)."""
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    shapes = [("a", 512, 1024, 4096), ("b", 512, 4096, 1024), ("c", 300, 1160, 776), ("d", 2048, 512, 1024)]
    ps = [synth.make_problem(n, T, o, i, 100 + k) for k, (n, T, o, i) in enumerate(shapes)]
    if mode == "int8":
        ps = [p for p in ps if p.inn % 256 == 0]
    if mode == "fp8":
        ps = [p for p in ps if p.inn % 16 == 0]

    def fresh():
        out = []
        for p in ps:
            d = dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone())
            if mode == "bf16":
                d["m"], d["v"] = p.m.to(torch.bfloat16).to(DEV), p.v.to(torch.bfloat16).to(DEV)
            elif mode == "int8":
                mq, ms, vq, vs = fo.quantize(p.m.numpy(), p.v.numpy())
                d.update(m=torch.from_numpy(mq).to(DEV), v=torch.from_numpy(vq).to(DEV),
                         m_scale=torch.from_numpy(ms).to(DEV), v_scale=torch.from_numpy(vs).to(DEV))
            elif mode == "fp8":
                mq, ms = fo.fp8_quantize(p.m.numpy())
                vq, vs = fo.fp8_quantize(p.v.numpy())
                d.update(m=torch.from_numpy(mq).to(DEV), v=torch.from_numpy(vq).to(DEV),
                         m_scale=torch.from_numpy(ms).to(DEV), v_scale=torch.from_numpy(vs).to(DEV))
            out.append(d)
        return out

    def run(L):
        if mode in ("fp32", "bf16", "int8", "fp8"):
            fb.forge_wgrad_adamw_grouped(L, 10, *hpt, {"fp32": fb.FP32, "bf16": fb.BF16, "int8": fb.INT8, "fp8": fb.FP8}[mode])
        elif mode == "sr":
            fb.forge_wgrad_adamw_sr_grouped(L, 10, *hpt, fb.FP32, 99)
        elif mode == "momentum":
            fb.forge_wgrad_step_grouped([dict(d, v=None) for d in L], "momentum", 3, 1e-2, momentum=0.9)
        elif mode == "sgd":
            fb.forge_wgrad_step_grouped([dict(d, m=None, v=None) for d in L], "sgd", 3, 1e-2)
        else:
            fb.forge_wgrad_accumulate_grouped([dict(X=d["X"], dY=d["dY"], W=None, m=d["m"], v=None) for d in L], 0.9)

    ref = None
    for _ in range(8):
        L = fresh()
        run(L)
        torch.cuda.synchronize()
        snap = [[d[k].clone() for k in ("W", "m", "v", "m_scale", "v_scale") if d.get(k) is not None] for d in L]
        if ref is None:
            ref = snap
        else:
            assert all(torch.equal(x, y) for a, b in zip(ref, snap) for x, y in zip(a, b)), mode


def test_grouped_host_entry_fp8_matches_device_path_bitwise():
    """forge_wgrad_adamw_grouped_host with FP8 moments: codes, W and both scale / amax pairs equal the device-resident call."""
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    ps = [synth.make_problem("a", 200, 136, 272, 71), synth.make_problem("b", 96, 256, 512, 72)]
    host, devs = [], []
    for p in ps:
        mq, ms = fo.fp8_quantize(p.m.numpy())
        vq, vs = fo.fp8_quantize(p.v.numpy())
        t = dict(X=p.X, dY=p.dY, W=p.W.clone(), m=torch.from_numpy(mq.copy()), v=torch.from_numpy(vq.copy()),
                 m_scale=torch.from_numpy(ms.copy()), v_scale=torch.from_numpy(vs.copy()))
        host.append({k: x.clone().pin_memory() for k, x in t.items()})
        devs.append({k: x.to(DEV).clone() for k, x in t.items()})
    fb.forge_wgrad_adamw_grouped_host(host, 10, *hpt, fb.FP8)
    fb.forge_wgrad_adamw_grouped(devs, 10, *hpt, fb.FP8)
    torch.cuda.synchronize()
    for h, d, p in zip(host, devs, ps):
        for k in ("W", "m", "v", "m_scale", "v_scale"):
            assert torch.equal(h[k], d[k].cpu()), k
        assert not torch.equal(h["W"], p.W) and float(h["m_scale"][1]) > 0.0


# ------------------------------------------------------------------ DP schedules ------
@pytest.mark.parametrize("moment", ["fp32", "int8"])
def test_dp_bucket_schedule_single_rank_is_bitwise_the_fused_step(moment):
    """dp.bucket_step_adamw with the library's own steps (store-G into a rotating bucket -> update from the bucket),
    buckets that cut problems into row ranges and mix pieces of two problems: at world size 1 and one micro-batch it
    must be bit-identical to the fused call (Prop. 1 bucket-wise)."""
    from paper_2606_22932_b200 import dp
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    shapes = [(384, 512), (200, 256), (640, 768)]
    fused, bucketed = [], []
    for i, (o, c) in enumerate(shapes):
        p = synth.make_problem(f"dp{i}", 300, o, c, 90 + i)
        d = dict(X=p.X.to(DEV), dY=p.dY.to(DEV), W=p.W.to(DEV).clone())
        if moment == "fp32":
            d.update(m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone())
        else:
            mq, ms, vq, vs = fo.quantize(p.m.numpy(), p.v.numpy())
            d.update(m=torch.from_numpy(mq.copy()).to(DEV), v=torch.from_numpy(vq.copy()).to(DEV),
                     m_scale=torch.from_numpy(ms.copy()).to(DEV), v_scale=torch.from_numpy(vs.copy()).to(DEV))
        fused.append(d)
        bucketed.append({k: (t if k in ("X", "dY") else t.clone()) for k, t in d.items()})
    plan = dp.BucketPlan(shapes, 4 * 256 * 768, slots=2)
    assert len(plan.buckets) >= 3 and any(len(b) > 1 for b in plan.buckets)
    pool = [torch.full((plan.slot_elems,), float("nan"), device=DEV) for _ in range(plan.slots)]
    dp.bucket_step_adamw(bucketed, 10, hpt, plan, pool)
    fb.forge_wgrad_adamw_grouped(fused, 10, *hpt, fb.FP32 if moment == "fp32" else fb.INT8)
    torch.cuda.synchronize()
    for a, b in zip(bucketed, fused):
        for k in a:
            assert torch.equal(a[k].view(torch.uint8), b[k].view(torch.uint8)), k
    assert plan.transient_bytes < sum(o * c for o, c in shapes) * 4


def test_dp_micro_batch_accumulation_and_reduce_into_state_against_the_oracle():
    """Two micro-batches summed in the fp32 bucket (store-G, then accumulate with mu = 1) before the update, and the
    single-rank reduce-into-state B <- mu*B + dY^T X; both against the oracle on all tokens."""
    from paper_2606_22932_b200 import dp
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    T, o, c = 256, 384, 512
    p = synth.make_problem("mb", T, o, c, 99)
    d = dict(X=[p.X[:96].to(DEV), p.X[96:].to(DEV)], dY=[p.dY[:96].to(DEV), p.dY[96:].to(DEV)],
             W=p.W.to(DEV).clone(), m=p.m.to(DEV).clone(), v=p.v.to(DEV).clone())
    plan = dp.BucketPlan([(o, c)], 4 * 128 * c, slots=2)
    pool = [torch.empty(plan.slot_elems, device=DEV) for _ in range(plan.slots)]
    dp.bucket_step_adamw([d], 10, hpt, plan, pool)
    B = dict(X=p.X.to(DEV), dY=p.dY.to(DEV), m=p.m.to(DEV).clone())
    dp.reduce_into_state([B], 0.9)
    torch.cuda.synchronize()
    G, E = fo.wgrad(synth.bf16_bits(p.dY), synth.bf16_bits(p.X), with_abs=True)
    Wo, mo, vo = synth.bf16_bits(p.W).copy(), p.m.numpy().copy(), p.v.numpy().copy()
    fo.adamw_fp32(Wo, mo, vo, G, 10, *hpt)
    e = T * 2.0 ** -23 * E
    mg, vg = d["m"].cpu().numpy().astype(np.float64), d["v"].cpu().numpy().astype(np.float64)
    assert (np.abs(mg - mo) <= 1e-4 * np.abs(mo) + (1 - hp["beta1"]) * e).all()
    assert (np.abs(vg - vo) <= 1e-4 * vo + (1 - hp["beta2"]) * (2 * np.abs(G) * e + e * e)).all()
    assert float((synth.bf16_bits(d["W"].cpu()) == Wo).mean()) > 0.99
    Bo = p.m.numpy().copy()
    fo.accumulate(Bo, G, 0.9)
    assert (np.abs(B["m"].cpu().numpy().astype(np.float64) - Bo) <= e + 2.0 ** -22 * np.abs(Bo)).all()


@pytest.mark.parametrize("moment", ["fp32", "int8", "fp8"])
def test_grouped_host_entry_row_slices_are_bitwise_the_device_call(moment):
    """forge_wgrad_adamw_grouped_host streams a problem's state in ~64 MB row slices (several slices and a ragged last
    one here: 2400 rows of 8192 columns); the slices are whole tile rows reading a column slice of the resident dY, so
    the result equals the device-resident call bit for bit, scales / amax included."""
    hp = synth.HP_DEFAULT
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    p = synth.make_problem("big", 64, 2400, 8192, 81)
    t = dict(X=p.X, dY=p.dY, W=p.W.clone())
    if moment == "fp32":
        t.update(m=p.m.clone(), v=p.v.clone())
    elif moment == "int8":
        mq, ms, vq, vs = fo.quantize(p.m.numpy(), p.v.numpy())
        t.update(m=torch.from_numpy(mq.copy()), v=torch.from_numpy(vq.copy()), m_scale=torch.from_numpy(ms.copy()),
                 v_scale=torch.from_numpy(vs.copy()))
    else:
        mq, ms = fo.fp8_quantize(p.m.numpy())
        vq, vs = fo.fp8_quantize(p.v.numpy())
        t.update(m=torch.from_numpy(mq.copy()), v=torch.from_numpy(vq.copy()), m_scale=torch.from_numpy(ms.copy()),
                 v_scale=torch.from_numpy(vs.copy()))
    small = synth.make_problem("small", 64, 136, 272, 82)       # a second, single-slice problem in the same call
    t2 = dict(X=small.X, dY=small.dY, W=small.W.clone())
    if moment == "fp32":
        t2.update(m=small.m.clone(), v=small.v.clone())
    elif moment == "int8":
        t2 = None                                               # int8 needs in % 256 == 0
    else:
        mq, ms = fo.fp8_quantize(small.m.numpy())
        vq, vs = fo.fp8_quantize(small.v.numpy())
        t2.update(m=torch.from_numpy(mq.copy()), v=torch.from_numpy(vq.copy()), m_scale=torch.from_numpy(ms.copy()),
                  v_scale=torch.from_numpy(vs.copy()))
    ts = [t] + ([t2] if t2 is not None else [])
    host = [{k: x.clone().pin_memory() for k, x in d.items()} for d in ts]
    devs = [{k: x.to(DEV).clone() for k, x in d.items()} for d in ts]
    mdt = {"fp32": fb.FP32, "int8": fb.INT8, "fp8": fb.FP8}[moment]
    fb.forge_wgrad_adamw_grouped_host(host, 10, *hpt, mdt)
    fb.forge_wgrad_adamw_grouped(devs, 10, *hpt, mdt)
    torch.cuda.synchronize()
    for h, d, src in zip(host, devs, ts):
        for k in h:
            assert torch.equal(h[k].view(torch.uint8), d[k].cpu().view(torch.uint8)), k
        assert not torch.equal(h["W"], src["W"])

"""Pins for oracle/forge_oracle_families.c (the other coordinate-wise families of PAPER.md:267 Def. 1):
each rule is checked against torch.optim on CPU in float64 -- a library call with injected state, the
paper's own method of verification -- over several consecutive steps, and Lion (not in
torch.optim) against its closed forms.  The oracle's W is bf16; the comparison is made on its unrounded
fp64 W' (debug output) and on fp32 state, chained through the oracle's own rounded values."""
import numpy as np
import pytest
import torch

from oracle import forge_oracle as fo

OUT, IN = 48, 64


def bf16_bits(x: np.ndarray) -> np.ndarray:
    return fo.f64_to_bf16(x.astype(np.float64))


def torch_reference(family, hp):
    p = torch.nn.Parameter(torch.zeros(OUT, IN, dtype=torch.float64))
    if family == "sgd":
        return p, torch.optim.SGD([p], lr=hp["lr"], weight_decay=hp["wd"])
    if family == "momentum":
        return p, torch.optim.SGD([p], lr=hp["lr"], weight_decay=hp["wd"], momentum=hp["momentum"], nesterov=hp["nesterov"])
    if family == "rmsprop":
        return p, torch.optim.RMSprop([p], lr=hp["lr"], alpha=hp["beta2"], eps=hp["eps"], weight_decay=hp["wd"])
    if family == "adagrad":
        return p, torch.optim.Adagrad([p], lr=hp["lr"], eps=hp["eps"], weight_decay=hp["wd"])
    if family == "adamax":
        return p, torch.optim.Adamax([p], lr=hp["lr"], betas=(hp["beta1"], hp["beta2"]), eps=hp["eps"], weight_decay=hp["wd"])
    if family == "nadam":
        return p, torch.optim.NAdam([p], lr=hp["lr"], betas=(hp["beta1"], hp["beta2"]), eps=hp["eps"], weight_decay=hp["wd"])
    if family == "radam":
        return p, torch.optim.RAdam([p], lr=hp["lr"], betas=(hp["beta1"], hp["beta2"]), eps=hp["eps"], weight_decay=hp["wd"])
    raise KeyError(family)


STATE_KEYS = {"momentum": ["momentum_buffer"], "rmsprop": ["square_avg"], "adagrad": ["sum"],
              "adamax": ["exp_avg", "exp_inf"], "nadam": ["exp_avg", "exp_avg_sq"], "radam": ["exp_avg", "exp_avg_sq"]}


@pytest.mark.parametrize("family,extra", [
    ("sgd", {}), ("momentum", {"momentum": 0.9}), ("momentum", {"momentum": 0.8, "nesterov": True}),
    ("rmsprop", {"beta2": 0.99}), ("adagrad", {"eps": 1e-10}), ("adamax", {}), ("nadam", {}), ("radam", {})])
def test_family_matches_torch_optim_float64_over_eight_steps(family, extra):
    """Steps 1..8 cover RAdam's un-rectified (rho_t <= 5, t <= 5 at beta2 = 0.999) and rectified branches."""
    hp = dict(lr=1e-2, beta1=np.float32(0.9).item(), beta2=np.float32(0.999).item(), eps=1e-8, wd=0.05, momentum=0.0, nesterov=False)
    hp.update({k: (np.float32(v).item() if isinstance(v, float) else v) for k, v in extra.items()})
    hp["lr"], hp["eps"], hp["wd"] = (np.float32(hp[k]).item() for k in ("lr", "eps", "wd"))   # the ABI carries floats
    rng = np.random.default_rng(11)
    W = bf16_bits(rng.normal(0, 0.02, (OUT, IN)))
    ns = fo.FAMILY_STATES[family]
    states = [np.zeros((OUT, IN), np.float32) for _ in range(ns)]
    p, opt = torch_reference(family, hp)
    for step in range(1, 9):
        G = rng.normal(0, 1e-2, (OUT, IN))
        # torch starts every step from the oracle's (rounded) W and state: one-step comparison, chained inputs
        with torch.no_grad():
            p.copy_(torch.from_numpy(fo.bf16_to_f64(W)))
        p.grad = torch.from_numpy(G.copy())
        if step > 1:
            for key, s in zip(STATE_KEYS.get(family, []), states):
                opt.state[p][key].copy_(torch.from_numpy(s.astype(np.float64)))
        opt.step()
        Wd = fo.family_step(family, W, *(states + [None] * (2 - ns)), G, step, hp["lr"], hp["beta1"], hp["beta2"],
                            hp["eps"], hp["wd"], hp["momentum"], hp["nesterov"], debug=True)
        ref = p.detach().numpy()
        # torch.optim.NAdam keeps mu_product in a float32 scalar tensor: 1e-7 relative on the step size
        atol = 1e-6 * hp["lr"] if family == "nadam" else 1e-15
        assert np.allclose(Wd, ref, rtol=1e-12, atol=atol), (family, step, np.abs(Wd - ref).max())
        assert np.array_equal(W, fo.f64_to_bf16(Wd))                         # one RNE rounding of the fp64 W'
        for key, s in zip(STATE_KEYS.get(family, []), states):
            t = opt.state[p][key].numpy()
            assert np.allclose(s, t, rtol=2e-7, atol=1e-30), (family, key, step)     # fp32 storage of the fp64 state


def test_lion_closed_forms_and_bruteforce():
    rng = np.random.default_rng(5)
    lr, b1, b2, wd = (np.float32(x).item() for x in (1e-4, 0.9, 0.99, 0.1))
    Wf = rng.normal(0, 0.02, (OUT, IN))
    W0 = bf16_bits(Wf)
    m0 = rng.normal(0, 1e-3, (OUT, IN)).astype(np.float32)
    G = rng.normal(0, 1e-3, (OUT, IN))
    G[0, :4] = 0.0
    m0[0, :4] = 0.0                                                         # sign(0) = 0: decay only
    W, m = W0.copy(), m0.copy()
    Wd = fo.family_step("lion", W, m, None, G, 1, lr, b1, b2, 0.0, wd, debug=True)
    w = fo.bf16_to_f64(W0)
    for i in range(OUT):                                                    # Chen et al. 2023 Alg. 2, coordinate by coordinate
        for j in range(IN):
            c = b1 * float(m0[i, j]) + (1 - b1) * G[i, j]
            s = 1.0 if c > 0 else (-1.0 if c < 0 else 0.0)
            assert Wd[i, j] == w[i, j] * (1 - lr * wd) - lr * s
            assert m[i, j] == np.float32(b2 * float(m0[i, j]) + (1 - b2) * G[i, j])
    assert np.all(Wd[0, :4] == w[0, :4] * (1 - lr * wd))
    # every non-degenerate coordinate moves by exactly lr (plus decay): |dW + lr*wd*w| == lr
    moved = np.abs(Wd - w * (1 - lr * wd))
    assert np.allclose(moved[1:], lr, rtol=1e-12)
    # beta1 = beta2 = 0: direction is sign(g), state becomes g
    W, m = W0.copy(), m0.copy()
    Wd = fo.family_step("lion", W, m, None, G, 1, lr, 0.0, 0.0, 0.0, 0.0, debug=True)
    assert np.array_equal(Wd, w - lr * np.sign(G)) and np.array_equal(m, G.astype(np.float32))


def test_families_reduce_to_each_other_and_bf16_state():
    rng = np.random.default_rng(9)
    W0 = bf16_bits(rng.normal(0, 0.02, (OUT, IN)))
    G = rng.normal(0, 1e-2, (OUT, IN))
    lr = np.float32(1e-2).item()
    # momentum with mu = 0 is SGD; lr = 0 leaves W untouched while state moves
    Wa, Wb = W0.copy(), W0.copy()
    buf = np.zeros((OUT, IN), np.float32)
    fo.family_step("sgd", Wa, None, None, G, 3, lr, wd=0.0)
    fo.family_step("momentum", Wb, buf, None, G, 3, lr, wd=0.0, momentum=0.0)
    assert np.array_equal(Wa, Wb) and np.array_equal(buf, G.astype(np.float32))
    Wc, s = W0.copy(), np.zeros((OUT, IN), np.float32)
    fo.family_step("adagrad", Wc, s, None, G, 1, 0.0)
    assert np.array_equal(Wc, W0) and np.array_equal(s, (G * G).astype(np.float32))
    # bf16 state: same rule, state rounded RNE on store, W' from the unrounded state (reading S3)
    W32, W16 = W0.copy(), W0.copy()
    s32 = np.full((OUT, IN), 1e-4, np.float32)
    s16 = fo.f64_to_bf16(s32.astype(np.float64))
    s32 = fo.bf16_to_f64(s16).astype(np.float32)
    fo.family_step("rmsprop", W32, s32, None, G, 2, lr, beta2=np.float32(0.99).item())
    fo.family_step("rmsprop", W16, s16, None, G, 2, lr, beta2=np.float32(0.99).item())
    assert np.array_equal(W32, W16) and np.array_equal(s16, fo.f64_to_bf16(s32.astype(np.float64)))


def test_accumulate_into_state_is_addmm_with_beta():
    """B <- mu B + dY^T X "through the GEMM's own beta" == torch.addmm(B, dY^T, X, beta=mu)."""
    rng = np.random.default_rng(21)
    T = 40
    dY = fo.f64_to_bf16(rng.normal(0, 1e-2, (T, OUT)))
    X = fo.f64_to_bf16(rng.normal(0, 1.0, (T, IN)))
    B0 = rng.normal(0, 1e-3, (OUT, IN)).astype(np.float32)
    mu = np.float32(0.95).item()
    B = B0.copy()
    fo.accumulate(B, fo.wgrad(dY, X), mu)
    ref = torch.addmm(torch.from_numpy(B0.astype(np.float64)), torch.from_numpy(fo.bf16_to_f64(dY)).t(),
                      torch.from_numpy(fo.bf16_to_f64(X)), beta=mu).numpy()
    assert np.allclose(B, ref, rtol=1e-7, atol=1e-12)
    # mu = 0 stores the gradient itself; G = 0 only decays; bf16 storage is one RNE rounding of the same value
    Bz = B0.copy()
    fo.accumulate(Bz, fo.wgrad(dY, X), 0.0)
    assert np.array_equal(Bz, fo.wgrad(dY, X).astype(np.float32))
    Bd = B0.copy()
    fo.accumulate(Bd, np.zeros((OUT, IN)), mu)
    assert np.array_equal(Bd, (mu * B0.astype(np.float64)).astype(np.float32))
    Bb = fo.f64_to_bf16(B0.astype(np.float64))
    exp = fo.f64_to_bf16(mu * fo.bf16_to_f64(Bb) + fo.wgrad(dY, X))
    fo.accumulate(Bb, fo.wgrad(dY, X), mu)
    assert np.array_equal(Bb, exp)


def test_stochastic_rounding_store_dead_zone_unbiasedness_and_bounds():
    """PAPER.md:1450 SR microcheck ("dead zone, unbiasedness": RNE drift 0.000, SR -8.195e-4 vs -8.0e-4 target):
    an update far below half a bf16 ulp never moves an RNE weight, while the SR weight drifts by the exact amount
    on average.  Plus: SR returns one of the two bf16 neighbours of x, exactly x when x is representable, and its
    up-probability is the fp32 fraction."""
    w0, delta, steps, n = 1.0, -8.0e-6, 100, 4096                 # bf16 ulp below 1.0 is 2^-8 = 3.9e-3 >> |delta|
    rne = fo.f64_to_bf16(np.full(n, w0))
    for _ in range(steps):
        rne = fo.f64_to_bf16(fo.bf16_to_f64(rne) + delta)
    assert np.all(fo.bf16_to_f64(rne) == w0)                       # dead zone: drift exactly 0
    sr = fo.f64_to_bf16(np.full(n, w0))
    for step in range(1, steps + 1):
        cur = fo.bf16_to_f64(sr)
        sr = np.array([fo.bf16_sr(cur[i] + delta, fo.sr_bits(1234, step, 0, i // 64, i % 64)) for i in range(n)], np.uint16)
    drift = float((fo.bf16_to_f64(sr) - w0).mean())
    target = steps * delta                                         # -8.0e-4, the paper's target
    sigma = np.sqrt(steps * abs(delta) * 2.0 ** -8 / n)            # binomial spread of the mean
    assert abs(drift - target) < 5 * sigma, (drift, target)
    # neighbours, exactness, probability
    rng = np.random.default_rng(0)
    for x in rng.normal(0, 1, 200):
        lo_hi = {int(fo.bf16_sr(x, 0)), int(fo.bf16_sr(x, 0xFFFF))}
        f = np.float32(x)
        trunc = int(f.view(np.uint32)) >> 16
        assert lo_hi <= {trunc, trunc + 1}
        frac = int(f.view(np.uint32)) & 0xFFFF
        ups = sum(int(fo.bf16_sr(x, r)) == trunc + 1 for r in range(0, 65536, 257))
        assert abs(ups / 256 - frac / 65536) < 0.01
    exact = float(fo.bf16_to_f64(fo.f64_to_bf16(np.array([0.7])))[0])
    assert all(fo.bf16_sr(exact, r) == int(fo.f64_to_bf16(np.array([exact]))[0]) for r in (0, 1, 0x8000, 0xFFFF))
    # the generator: 16 bits, depends on every key, roughly uniform
    base = fo.sr_bits(1, 2, 3, 4, 5)
    assert 0 <= base < 65536 and len({base, fo.sr_bits(2, 2, 3, 4, 5), fo.sr_bits(1, 3, 3, 4, 5), fo.sr_bits(1, 2, 4, 4, 5),
                                      fo.sr_bits(1, 2, 3, 5, 5), fo.sr_bits(1, 2, 3, 4, 6), fo.sr_bits(1 << 40, 2, 3, 4, 5)}) == 7
    bits = np.array([fo.sr_bits(9, 1, 0, r, c) for r in range(64) for c in range(64)])
    assert abs(bits.mean() / 65535 - 0.5) < 0.02 and abs((bits & 1).mean() - 0.5) < 0.03


def test_adamw_sr_equals_rne_oracle_up_to_the_final_rounding():
    rng = np.random.default_rng(4)
    W0 = bf16_bits(rng.normal(0, 0.02, (OUT, IN)))
    m0 = rng.normal(0, 1e-4, (OUT, IN)).astype(np.float32)
    v0 = np.abs(rng.normal(0, 1e-6, (OUT, IN))).astype(np.float32)
    G = rng.normal(0, 1e-2, (OUT, IN))
    hp = (np.float32(1e-3).item(), np.float32(0.9).item(), np.float32(0.999).item(), 1e-8, np.float32(0.1).item())
    Wr, mr, vr = W0.copy(), m0.copy(), v0.copy()
    Wd, _, _ = fo.adamw_fp32(Wr, mr, vr, G, 7, *hp, debug=True)
    Ws, ms, vs = W0.copy(), m0.copy(), v0.copy()
    fo.adamw_fp32_sr(Ws, ms, vs, G, 7, *hp, seed=99, stream=2)
    assert np.array_equal(ms, mr) and np.array_equal(vs, vr)       # only the store of W differs
    for i in range(0, OUT, 7):
        for j in range(0, IN, 5):
            assert int(Ws[i, j]) == fo.bf16_sr(Wd[i, j], fo.sr_bits(99, 7, 2, i, j))
    assert np.all(np.abs(Ws.astype(np.int32) - Wr.astype(np.int32)) <= 1)


def test_e4m3_codec_against_torch_float8_and_by_hand():
    """e4m3 (bias 7, 3 mantissa bits, max 448, subnormal grid 2^-9): every code decodes like torch.float8_e4m3fn;
    encoding matches torch's RNE cast wherever torch does not overflow; beyond 448 the oracle saturates (the
    hardware cvt.rn.satfinite; torch's cast returns NaN there)."""
    codes = torch.arange(256, dtype=torch.uint8)
    ref = codes.view(torch.float8_e4m3fn).float().numpy()
    mine = np.array([fo.e4m3_to_double(c) for c in range(256)])
    assert np.array_equal(np.isnan(ref), np.isnan(mine)) and np.array_equal(ref[~np.isnan(ref)], mine[~np.isnan(mine)])
    rng = np.random.default_rng(8)
    xs = np.concatenate([rng.normal(0, 100, 20000), rng.normal(0, 0.02, 20000), rng.uniform(-448, 448, 20000),
                         mine[~np.isnan(mine)], (mine[:-1] + mine[1:])[~np.isnan(mine[:-1] + mine[1:])] / 2]).astype(np.float32)
    xs = xs[np.abs(xs) <= 448]
    tref = torch.from_numpy(xs).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = np.array([fo.e4m3_from_float(x) for x in xs], np.uint8)
    nz = (tref & 0x7F) != 0                                   # +0 / -0 of tiny negatives: compare magnitudes only there
    assert np.array_equal(got[nz], tref[nz]) and np.all((got[~nz] & 0x7F) == 0)
    # by hand: ties to even on the subnormal grid, carry into the exponent, saturation, NaN
    assert fo.e4m3_from_float(2.0 ** -10) == 0 and fo.e4m3_from_float(1.5 * 2.0 ** -10) == 1
    assert fo.e4m3_from_float(3 * 2.0 ** -10) == 2                       # 1.5 grid units: tie -> even (2)
    assert fo.e4m3_from_float(1.9375) == 0x40 and fo.e4m3_from_float(1.0) == 0x38 and fo.e4m3_from_float(-1.0) == 0xB8
    assert fo.e4m3_from_float(448.0) == 0x7E and fo.e4m3_from_float(1e9) == 0x7E and fo.e4m3_from_float(-1e9) == 0xFE
    assert fo.e4m3_from_float(float("inf")) == 0x7E and (fo.e4m3_from_float(float("nan")) & 0x7F) == 0x7F


def test_fp8_quantiser_and_step_properties():
    rng = np.random.default_rng(12)
    x = rng.normal(0, 1e-4, (OUT, IN)).astype(np.float32)
    code, scale = fo.fp8_quantize(x)
    assert scale[0] == np.float32(np.abs(x).max() / np.float32(448.0))
    deq = fo.fp8_dequantize(code, scale)
    # relative error <= 2^-4 (3 mantissa bits) for normals, absolute <= half the subnormal grid below
    err = np.abs(deq - x)
    assert np.all(err <= np.maximum(np.abs(x) * 2.0 ** -4, 2.0 ** -10 * scale[0]) * 1.0001)
    assert (code.flatten()[np.abs(x).argmax()] & 0x7F) == 0x7E            # the absmax element maps to +-448
    # one AdamW step: consistent with the fp32-moment oracle started from the dequantised state
    W0 = bf16_bits(rng.normal(0, 0.02, (OUT, IN)))
    v0 = np.abs(rng.normal(0, 1e-6, (OUT, IN))).astype(np.float32)
    vq, vs = fo.fp8_quantize(v0)
    G = rng.normal(0, 1e-2, (OUT, IN))
    hp = (np.float32(1e-3).item(), np.float32(0.9).item(), np.float32(0.999).item(), 1e-8, np.float32(0.1).item())
    Wr = W0.copy(); mr = fo.fp8_dequantize(code, scale).astype(np.float32); vr = fo.fp8_dequantize(vq, vs).astype(np.float32)
    m_in, v_in = mr.astype(np.float64), vr.astype(np.float64)
    fo.adamw_fp32(Wr, mr, vr, G, 5, *hp)
    Wq, mq2, vq2, ms, vs2 = W0.copy(), code.copy(), vq.copy(), scale.copy(), vs.copy()
    fo.adamw_fp8(Wq, mq2, vq2, ms, vs2, G, 5, *hp)
    assert np.array_equal(Wq, Wr)                                        # W' comes from the unrounded m', v' (S3)
    assert ms[0] == scale[0] and np.isclose(ms[1], np.abs(mr).max(), rtol=1e-6) and np.isclose(vs2[1], vr.max(), rtol=1e-6)
    # stored m' = e4m3(m' / s): decoding recovers m' to 2^-4 relative (or saturates at 448 s when m' outgrew the old scale)
    mdeq = fo.fp8_dequantize(mq2, ms)
    lim = 448.0 * float(ms[0])
    ok = np.abs(mdeq - np.clip(mr, -lim, lim)) <= np.maximum(np.abs(mr) * 2.0 ** -4, 2.0 ** -10 * ms[0]) * 1.001
    assert ok.all()
    # delayed scaling: feeding the reported amax back gives a scale under which nothing saturates
    nxt = np.float32(ms[1] / np.float32(448.0))
    assert np.abs(mr).max() <= 448.0 * float(nxt) * (1 + 1e-6)

"""More oracle pins: the int8 blockwise quantiser against App. B's bounds, the
per-tile exactness claim (Prop. 1) and the qualitative ordering of App. E
(PAPER.md:349-362).  CPU only."""
import numpy as np
import torch

from oracle import forge_oracle as fo

HP = (1e-3, 0.9, 0.999, 1e-8, 0.1)
F = np.float32


def rand_bf16(rng, shape, sigma=1.0):
    x = torch.from_numpy((rng.standard_normal(shape) * sigma).astype(np.float32))
    return x.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16).copy()


def test_quantiser_error_bound_extremal_codes_and_floor():
    rng = np.random.default_rng(11)
    out, inn = 24, 1024
    m = (rng.standard_normal((out, inn)) * 1e-4).astype(F)
    v = ((rng.standard_normal((out, inn)) * 1e-3) ** 2).astype(F)
    mq, ms, vq, vs = fo.quantize(m, v)
    mb, vb = m.reshape(out, -1, 256), v.reshape(out, -1, 256)
    # stored scale = block absmax (fp32), S5
    assert np.array_equal(ms, np.abs(mb).max(-1)) and np.array_equal(vs, vb.max(-1))
    # |dequant(quant(x)) - x| <= s/2, s = a/127 resp. a/255
    sm = np.repeat(ms.astype(np.float64) / 127, 256, 1)
    sv = np.repeat(vs.astype(np.float64) / 255, 256, 1)
    assert (np.abs(fo.dequantize_m(mq, ms) - m) <= sm * (0.5 + 1e-6)).all()
    dv = fo.dequantize_v(vq, vs) - v
    floored = (vq == 1) & (v < 0.5 * sv)           # entries raised by the floor (S6)
    assert (np.abs(dv)[~floored] <= sv[~floored] * (0.5 + 1e-6)).all()
    assert (dv[floored] > 0).all() and (dv[floored] <= sv[floored]).all()
    assert floored.mean() > 0.01                    # the floor is not a corner case
    # the block maximum maps to +-127 / 255 exactly; ranges respected; v codes >= 1
    arg = np.abs(mb).argmax(-1)
    top = np.take_along_axis(mq.reshape(out, -1, 256), arg[..., None], -1)[..., 0]
    assert np.array_equal(np.abs(top.astype(int)), np.full_like(top, 127, dtype=int))
    assert np.array_equal(np.sign(top), np.sign(np.take_along_axis(mb, arg[..., None], -1)[..., 0]))
    assert (vq.reshape(out, -1, 256).max(-1) == 255).all() and vq.min() >= 1
    assert mq.min() >= -127 and mq.max() <= 127


def test_quantiser_zero_block_and_idempotence():
    rng = np.random.default_rng(12)
    m = (rng.standard_normal((4, 512)) * 1e-4).astype(F)
    v = np.abs(rng.standard_normal((4, 512)) * 1e-6).astype(F)
    m[1, 256:] = 0
    v[1, 256:] = 0
    mq, ms, vq, vs = fo.quantize(m, v)
    assert ms[1, 1] == 0 and vs[1, 1] == 0 and not mq[1, 256:].any() and not vq[1, 256:].any()
    assert not fo.dequantize_m(mq, ms)[1, 256:].any() and not fo.dequantize_v(vq, vs)[1, 256:].any()
    # quantising an already-dequantised block returns the same codes; scale within 1 fp32 ulp
    mq2, ms2, vq2, vs2 = fo.quantize(fo.dequantize_m(mq, ms), fo.dequantize_v(vq, vs))
    assert np.array_equal(mq, mq2) and np.array_equal(vq, vq2)
    assert np.allclose(ms, ms2, rtol=2e-7, atol=0) and np.allclose(vs, vs2, rtol=2e-7, atol=0)


def test_quantiser_hand_block():
    """A block small enough to do by hand: x_i = i/2 for i = -127..127 has a = 63.5, s = 0.5, so
    code_i = i exactly; v_i = i for i = 0..255 has a = 255, code_i = max(i, 1)."""
    m = np.zeros((1, 256)); m[0, :255] = np.arange(-127, 128) / 2.0
    v = np.arange(256, dtype=np.float64)[None, :]
    mq, ms, vq, vs = fo.quantize(m, v)
    assert ms[0, 0] == 63.5 and vs[0, 0] == 255.0
    assert np.array_equal(mq[0, :255], np.arange(-127, 128)) and mq[0, 255] == 0
    assert np.array_equal(vq[0], np.maximum(np.arange(256), 1))
    # ties to even (S7): x = 2.5 * s -> code 2, x = 3.5 * s -> code 4
    m = np.zeros((1, 256)); m[0, 0] = 127.0; m[0, 1] = 2.5; m[0, 2] = 3.5; m[0, 3] = -2.5
    mq, _, _, _ = fo.quantize(m, None)
    assert list(mq[0, :4]) == [127, 2, 4, -2]


def test_int8_step_consistent_with_fp32_step_on_dequantised_state():
    """The int8 mode is 'the same update' on the dequantised state (arithmetic and
    gradient stay fp32/unquantised); its unrounded outputs must equal the fp32-moment oracle fed
    with the dequantised moments, and W must be identical."""
    rng = np.random.default_rng(13)
    out, inn = 8, 512
    W0 = rand_bf16(rng, (out, inn), 0.02)
    m = (rng.standard_normal((out, inn)) * 1e-4).astype(F)
    v = np.abs(rng.standard_normal((out, inn)) * 1e-6).astype(F)
    G = rng.standard_normal((out, inn)) * 1e-2
    mq, ms, vq, vs = fo.quantize(m, v)
    mq_in, ms_in, vq_in, vs_in = mq.copy(), ms.copy(), vq.copy(), vs.copy()
    md0, vd0 = fo.dequantize_m(mq, ms), fo.dequantize_v(vq, vs)
    W1 = W0.copy()
    Wd1, md1, vd1 = fo.adamw_int8(W1, mq, vq, ms, vs, G, 10, *HP, debug=True)
    # reference: same formula through numpy in fp64 on the dequantised state
    b1, b2, lr, eps, wd = (float(F(x)) for x in (0.9, 0.999, 1e-3, 1e-8, 0.1))
    mref = b1 * md0 + (1 - b1) * G
    vref = b2 * vd0 + (1 - b2) * G * G
    assert np.allclose(md1, mref, rtol=1e-15, atol=0) and np.allclose(vd1, vref, rtol=1e-15, atol=0)
    # the stored state is the quantisation of the unrounded m', v'
    mq2, ms2, vq2, vs2 = fo.quantize(md1, vd1)
    assert np.array_equal(mq, mq2) and np.array_equal(vq, vq2)
    assert np.array_equal(ms, ms2) and np.array_equal(vs, vs2)
    assert np.array_equal(W1, fo.f64_to_bf16(Wd1))
    # and against an independent scale-index restatement: dequantise with numpy indexing, one coordinate at a time
    bc1, bc2 = 1 - b1 ** 10, 1 - b2 ** 10
    for (p_, q_) in [(0, 0), (3, 255), (3, 256), (7, 511), (5, 300)]:
        mm = float(mq_in[p_, q_]) * (float(ms_in[p_, q_ // 256]) / 127.0)
        vv = float(vq_in[p_, q_]) * (float(vs_in[p_, q_ // 256]) / 255.0)
        m1 = b1 * mm + (1 - b1) * G[p_, q_]
        v1 = b2 * vv + (1 - b2) * G[p_, q_] ** 2
        w1 = (1 - lr * wd) * fo.bf16_to_f64(W0)[p_, q_] - lr * (m1 / bc1) / (np.sqrt(v1 / bc2) + eps)
        assert abs(Wd1[p_, q_] - w1) <= 4e-16 * max(abs(w1), 1e-300) + 1e-18


def test_int8_weight_equals_fp32_oracle_on_dequantised_state_bitwise():
    """Pin of W' (and the unrounded m', v') of ``adamw_int8``: with block maxima 127 * 2^-20 (m) and 255 * 2^-30
    (v) the steps a/127 and a/255 are powers of two, every dequantised moment is an fp32 number, and the
    fp32-moment oracle -- pinned on its own against torch.optim.AdamW and the step-1 closed form -- can be fed
    the dequantised state exactly.  Both must then agree on W bit for bit and on the fp64 W', m', v' exactly
    (same update, only the storage differs).  A wrong scale index, a swapped m / v scale or a
    missing dequantisation step fails here."""
    rng = np.random.default_rng(131)
    out, inn = 6, 768
    W0 = rand_bf16(rng, (out, inn), 0.02)
    am, av = 127.0 * 2.0 ** -20, 255.0 * 2.0 ** -30
    m = np.clip(rng.standard_normal((out, inn)) * 3e-5, -0.99 * am, 0.99 * am)
    v = np.clip(np.abs(rng.standard_normal((out, inn))) * 6e-8, 0, 0.99 * av)
    # different maxima per block so that a wrong block index shows: block b of row p gets am * 2^-(p+b)
    for p_ in range(out):
        for b_ in range(inn // 256):
            k = 2.0 ** -((p_ + b_) % 4)
            m[p_, b_ * 256:(b_ + 1) * 256] *= k; v[p_, b_ * 256:(b_ + 1) * 256] *= k
            m[p_, b_ * 256 + (7 * p_ + b_) % 256] = -am * k if (p_ + b_) % 2 else am * k
            v[p_, b_ * 256 + (11 * p_ + 3 * b_) % 256] = av * k
    G = rng.standard_normal((out, inn)) * 1e-2
    mq, ms, vq, vs = fo.quantize(m, v)
    md0, vd0 = fo.dequantize_m(mq, ms), fo.dequantize_v(vq, vs)
    mf, vf = md0.astype(F), vd0.astype(F)
    assert np.array_equal(mf.astype(np.float64), md0) and np.array_equal(vf.astype(np.float64), vd0)
    assert len(np.unique(ms)) == 4 and len(np.unique(vs)) == 4
    W1, Wf = W0.copy(), W0.copy()
    Wd1, md1, vd1 = fo.adamw_int8(W1, mq, vq, ms, vs, G, 10, *HP, debug=True)
    Wdf, mdf, vdf = fo.adamw_fp32(Wf, mf, vf, G, 10, *HP, debug=True)
    assert np.array_equal(W1, Wf)
    assert np.array_equal(Wd1, Wdf) and np.array_equal(md1, mdf) and np.array_equal(vd1, vdf)


def test_prop1_tile_by_tile_equals_one_shot_bitwise():
    """Prop. 1: stepping tile by tile over any partition of the weight index
    set equals forming the full gradient and stepping once -- here bit for bit, because each
    coordinate's token sum runs in the same ascending order."""
    rng = np.random.default_rng(14)
    T, out, inn = 50, 48, 80
    dY, X = rand_bf16(rng, (T, out), 1e-2), rand_bf16(rng, (T, inn))
    W0 = rand_bf16(rng, (out, inn), 0.02)
    m0 = (rng.standard_normal((out, inn)) * 1e-4).astype(F)
    v0 = np.abs(rng.standard_normal((out, inn)) * 1e-6).astype(F)
    W, m, v = W0.copy(), m0.copy(), v0.copy()
    fo.adamw_fp32(W, m, v, fo.wgrad(dY, X), 3, *HP)
    Wt, mt, vt = W0.copy(), m0.copy(), v0.copy()
    row_cuts, col_cuts = [0, 16, 21, 48], [0, 32, 33, 80]      # ragged, uneven tiles
    for r0, r1 in zip(row_cuts[:-1], row_cuts[1:]):
        for c0, c1 in zip(col_cuts[:-1], col_cuts[1:]):
            Gt = fo.wgrad(np.ascontiguousarray(dY[:, r0:r1]), np.ascontiguousarray(X[:, c0:c1]))
            w, a, b = (np.ascontiguousarray(z[r0:r1, c0:c1]) for z in (Wt, mt, vt))
            fo.adamw_fp32(w, a, b, Gt, 3, *HP)
            Wt[r0:r1, c0:c1], mt[r0:r1, c0:c1], vt[r0:r1, c0:c1] = w, a, b
    assert np.array_equal(W, Wt) and np.array_equal(m, mt) and np.array_equal(v, vt)


def test_appendix_e_ordering_fp32_gradient_beats_bf16_rounded_gradient():
    """App. E / App. B: over 20 steps the path that feeds the optimizer
    the unrounded gradient tracks an all-fp64 reference more closely than the path that rounds G
    to bf16 first.  The printed digits (5.825e-4 vs 6.091e-4) are parity-unpinned (inputs not
    given); the state error, which the bf16 rounding of G drives directly, is the robust check."""
    rng = np.random.default_rng(15)
    T, out, inn, steps = 64, 64, 256, 20
    W0 = rand_bf16(rng, (out, inn), 0.02)
    Wf, mf, vf = W0.copy(), np.zeros((out, inn), F), np.zeros((out, inn), F)       # fused: fp64->fp32 G
    Ws, ms_, vs_ = W0.copy(), np.zeros((out, inn), F), np.zeros((out, inn), F)     # standard: bf16 G
    p = torch.nn.Parameter(torch.from_numpy(fo.bf16_to_f64(W0)))                  # never rounded
    opt = torch.optim.AdamW([p], lr=float(F(1e-3)), betas=(float(F(0.9)), float(F(0.999))),
                            eps=float(F(1e-8)), weight_decay=float(F(0.1)))
    for t in range(1, steps + 1):
        dY, X = rand_bf16(rng, (T, out), 1e-2), rand_bf16(rng, (T, inn))
        G = fo.wgrad(dY, X)
        fo.adamw_fp32(Wf, mf, vf, G, t, *HP)
        fo.adamw_fp32(Ws, ms_, vs_, fo.bf16_to_f64(fo.f64_to_bf16(G)), t, *HP)
        p.grad = torch.from_numpy(G.copy())
        opt.step()
    m_ref = opt.state[p]["exp_avg"].numpy()
    err_f = np.sqrt(np.mean((mf - m_ref) ** 2)) / np.sqrt(np.mean(m_ref ** 2))
    err_s = np.sqrt(np.mean((ms_ - m_ref) ** 2)) / np.sqrt(np.mean(m_ref ** 2))
    assert err_f < 1e-6 and err_s > 1e-4 and err_f < err_s
    Wref = p.detach().numpy()
    rms = lambda W: np.sqrt(np.mean((fo.bf16_to_f64(W) - Wref) ** 2)) / np.sqrt(np.mean(Wref ** 2))
    # both are dominated by the per-step bf16 rounding of W, same order as the paper's ~6e-4
    assert 1e-4 < rms(Wf) < 1e-2 and 1e-4 < rms(Ws) < 1e-2

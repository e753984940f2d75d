"""Pins for the CPU oracle (oracle/forge_oracle.c): every check here compares the oracle with
something other than itself -- exact rational arithmetic, a closed form, a library routine, or
an invariant the paper states.  None of these need a GPU."""
from fractions import Fraction

import numpy as np
import pytest
import torch

from oracle import forge_oracle as fo

HP = dict(lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.1)
F = np.float32


def hp_args(step, **kw):
    h = {**HP, **kw}
    return (step, h["lr"], h["beta1"], h["beta2"], h["eps"], h["wd"])


def rand_bf16(rng, shape, sigma=1.0):
    x = torch.from_numpy((rng.standard_normal(shape) * sigma).astype(np.float32))
    return x.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16).copy()


# --------------------------------------------------------------------------- bf16 rounding ---
def test_bf16_rne_matches_torch_cast_on_float32_inputs():
    """S9 / PAPER.md:1292: RNE.  torch's CPU fp32->bf16 cast is the library routine."""
    rng = np.random.default_rng(1)
    x = np.concatenate([
        rng.standard_normal(200000).astype(F),
        (rng.standard_normal(50000) * 1e-30).astype(F),
        (rng.standard_normal(50000) * 1e30).astype(F),
        rng.integers(0, 2**32, 400000, dtype=np.uint64).astype(np.uint32).view(F),  # raw patterns
        np.array([0.0, -0.0, np.inf, -np.inf, 1.0, 1.00390625, 1.01171875, 3.3895314e38,
                  3.4028235e38, 1e-40, 9.18e-41, 4.6e-41, 1.17549435e-38], dtype=F),
    ])
    x = x[~np.isnan(x)]
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = fo.f64_to_bf16(x.astype(np.float64))
    assert np.array_equal(got, want)


def test_bf16_rne_ties_and_single_rounding():
    # exact ties in bf16: 1 + 2^-8 is halfway between 1 and 1+2^-7 -> even (1.0)
    assert fo.lib().forge_oracle_bf16_from_double(1.0 + 2.0**-8) == 0x3F80
    assert fo.lib().forge_oracle_bf16_from_double(1.0 + 3 * 2.0**-8) == 0x3F82
    # just above the tie by less than an fp32 ulp: a double-rounding implementation returns 0x3F80
    assert fo.lib().forge_oracle_bf16_from_double(1.0 + 2.0**-8 + 2.0**-30) == 0x3F81
    assert fo.lib().forge_oracle_bf16_from_double(-(1.0 + 2.0**-8 + 2.0**-30)) == 0xBF81
    # carry into the exponent, overflow, NaN, signed zero
    assert fo.lib().forge_oracle_bf16_from_double(1.99999) == 0x4000
    assert fo.lib().forge_oracle_bf16_from_double(3.4e38) == 0x7F80
    assert fo.lib().forge_oracle_bf16_from_double(-0.0) == 0x8000
    assert fo.lib().forge_oracle_bf16_from_double(float("nan")) & 0x7FFF > 0x7F80
    # round trip of every finite bf16 pattern is the identity
    bits = np.arange(0, 1 << 16, dtype=np.uint32).astype(np.uint16)
    finite = (bits & 0x7F80) != 0x7F80
    assert np.array_equal(fo.f64_to_bf16(fo.bf16_to_f64(bits[finite])), bits[finite])


# --------------------------------------------------------------------------- the gradient ----
def test_wgrad_exact_rational_bruteforce():
    """PAPER.md:253 G_pq = sum_t dY_tp X_tq.  bf16 values are dyadic rationals, so Python's
    Fraction gives the exact sum; the fp64 oracle must match it to the last bit here."""
    rng = np.random.default_rng(2)
    T, out, inn = 5, 3, 4
    dY, X = rand_bf16(rng, (T, out), 1e-2), rand_bf16(rng, (T, inn))
    G = fo.wgrad(dY, X)
    dYf, Xf = fo.bf16_to_f64(dY), fo.bf16_to_f64(X)
    for p in range(out):
        for q in range(inn):
            exact = sum(Fraction(float(dYf[t, p])) * Fraction(float(Xf[t, q])) for t in range(T))
            assert abs(Fraction(float(G[p, q])) - exact) <= abs(exact) * Fraction(1, 2**50)
    # a transposed operand or a swapped index cannot survive a non-square, asymmetric case:
    assert G.shape == (out, inn)


def test_wgrad_matches_library_matmul_and_invariants():
    rng = np.random.default_rng(3)
    T, out, inn = 96, 40, 72
    dY, X = rand_bf16(rng, (T, out), 1e-3), rand_bf16(rng, (T, inn))
    G, E = fo.wgrad(dY, X, with_abs=True)
    ref = fo.bf16_to_f64(dY).T @ fo.bf16_to_f64(X)              # library fp64 matmul
    assert np.allclose(G, ref, rtol=0, atol=1e-15 * np.abs(E).max())
    assert np.allclose(E, np.abs(fo.bf16_to_f64(dY)).T @ np.abs(fo.bf16_to_f64(X)), rtol=1e-14)
    assert (np.abs(G) <= E * (1 + 1e-12)).all()
    # additivity over a split of the token axis (Prop. 1, gradient correctness step)
    G1, G2 = fo.wgrad(dY[:37].copy(), X[:37].copy()), fo.wgrad(dY[37:].copy(), X[37:].copy())
    assert np.allclose(G, G1 + G2, rtol=0, atol=1e-15 * np.abs(E).max())
    # token permutation leaves G unchanged up to fp64 rounding; dY = 0 gives exactly 0
    perm = rng.permutation(T)
    assert np.allclose(G, fo.wgrad(dY[perm].copy(), X[perm].copy()), rtol=0, atol=1e-15 * E.max())
    assert not fo.wgrad(np.zeros_like(dY), X).any()
    # row-subset API is exact for its rows
    assert np.array_equal(fo.wgrad(dY, X, rows=(7, 19)), G[7:19])


# --------------------------------------------------------------------------- AdamW -----------
def test_adamw_step1_closed_form():
    """north_star: from zero state at t=1, dW = -lr*(g/(|g|+eps) + wd*W), m=(1-b1)g, v=(1-b2)g^2."""
    rng = np.random.default_rng(4)
    shape = (16, 32)
    W = rand_bf16(rng, shape, 0.02)
    G = rng.standard_normal(shape) * 1e-2
    G[0, :4] = 0.0
    m, v = np.zeros(shape, F), np.zeros(shape, F)
    W0 = fo.bf16_to_f64(W)
    Wd, md, vd = fo.adamw_fp32(W, m, v, G, *hp_args(1), debug=True)
    lr, b1, b2, eps, wd = (float(F(HP[k])) for k in ("lr", "beta1", "beta2", "eps", "wd"))
    want = W0 - lr * (G / (np.abs(G) + eps) + wd * W0)
    # the rounding of sqrt(g^2/(1-b2)*(1-b2)) limits the agreement to a few fp64 ulps of lr
    assert np.abs(Wd - want).max() < 1e-15
    assert np.allclose(md, (1 - b1) * G, rtol=1e-15, atol=0)
    assert np.allclose(vd, (1 - b2) * G * G, rtol=1e-15, atol=0)
    assert np.array_equal(W, fo.f64_to_bf16(Wd)) and np.array_equal(m, md.astype(F))


@pytest.mark.parametrize("step", [1, 2, 10, 1000])
def test_adamw_general_state_vs_torch_optim_float64(step):
    """The paper's own small-tensor check (D=512, BT=256) against the library."""
    rng = np.random.default_rng(5 + step)
    D, BT = 512, 256
    dY, X = rand_bf16(rng, (BT, D), 1e-3), rand_bf16(rng, (BT, D))
    W = rand_bf16(rng, (D, D), 0.02)
    m = (rng.standard_normal((D, D)) * 1e-4).astype(F)
    v = np.abs(rng.standard_normal((D, D)) * 1e-6).astype(F)
    G = fo.wgrad(dY, X)
    p = torch.nn.Parameter(torch.from_numpy(fo.bf16_to_f64(W)))
    opt = torch.optim.AdamW([p], lr=float(F(HP["lr"])), betas=(float(F(HP["beta1"])), float(F(HP["beta2"]))),
                            eps=float(F(HP["eps"])), weight_decay=float(F(HP["wd"])), foreach=False, fused=False)
    p.grad = torch.from_numpy(G.copy())
    opt.state[p] = {"step": torch.tensor(float(step - 1)), "exp_avg": torch.from_numpy(m.astype(np.float64)),
                    "exp_avg_sq": torch.from_numpy(v.astype(np.float64))}
    opt.step()
    Wd, md, vd = fo.adamw_fp32(W, m, v, G, *hp_args(step), debug=True)
    assert np.abs(Wd - p.detach().numpy()).max() < 1e-14
    assert np.allclose(md, opt.state[p]["exp_avg"].numpy(), rtol=1e-13, atol=1e-20)
    assert np.allclose(vd, opt.state[p]["exp_avg_sq"].numpy(), rtol=1e-13, atol=1e-26)


def test_adamw_special_cases():
    rng = np.random.default_rng(6)
    shape = (8, 64)
    W0 = rand_bf16(rng, shape, 0.02)
    m0 = (rng.standard_normal(shape) * 1e-4).astype(F)
    v0 = np.abs(rng.standard_normal(shape) * 1e-6).astype(F)
    G = rng.standard_normal(shape) * 1e-2
    b1, b2 = float(F(0.9)), float(F(0.999))
    # lr = 0: W unchanged while m, v move
    W, m, v = W0.copy(), m0.copy(), v0.copy()
    fo.adamw_fp32(W, m, v, G, *hp_args(7, lr=0.0))
    assert np.array_equal(W, W0) and not np.array_equal(m, m0) and not np.array_equal(v, v0)
    # g = 0: the decay-only case of Remark 1: m' = b1 m, v' = b2 v
    W, m, v = W0.copy(), m0.copy(), v0.copy()
    _, md, vd = fo.adamw_fp32(W, m, v, np.zeros(shape), *hp_args(7), debug=True)
    assert np.allclose(md, b1 * m0.astype(np.float64), rtol=1e-15) and np.allclose(vd, b2 * v0.astype(np.float64), rtol=1e-15)
    # b1 = b2 = 0: W' = (1-lr wd) W - lr g/(|g|+eps) at any t
    W, m, v = W0.copy(), m0.copy(), v0.copy()
    Wd, _, _ = fo.adamw_fp32(W, m, v, G, *hp_args(5, beta1=0.0, beta2=0.0), debug=True)
    lr, eps, wd = float(F(1e-3)), float(F(1e-8)), float(F(0.1))
    w = fo.bf16_to_f64(W0)
    assert np.abs(Wd - ((1 - lr * wd) * w - lr * G / (np.abs(G) + eps))).max() < 1e-16
    # wd = 0, g = 0, m = 0: W unchanged
    W = W0.copy()
    fo.adamw_fp32(W, np.zeros(shape, F), v0.copy(), np.zeros(shape), *hp_args(3, wd=0.0))
    assert np.array_equal(W, W0)
    # sign: a positive gradient from zero state moves W down
    W = W0.copy()
    fo.adamw_fp32(W, np.zeros(shape, F), np.zeros(shape, F), np.ones(shape), *hp_args(1, wd=0.0))
    assert (fo.bf16_to_f64(W) < fo.bf16_to_f64(W0)).all()


def test_bf16_moment_mode_is_same_update_with_rounded_state():
    rng = np.random.default_rng(7)
    shape = (8, 64)
    W0 = rand_bf16(rng, shape, 0.02)
    mb, vb = rand_bf16(rng, shape, 1e-4), rand_bf16(rng, shape, 1e-6) & 0x7FFF
    G = rng.standard_normal(shape) * 1e-2
    W1, m1, v1 = W0.copy(), fo.bf16_to_f64(mb).astype(F), fo.bf16_to_f64(vb).astype(F)
    Wd32, md32, vd32 = fo.adamw_fp32(W1, m1, v1, G, *hp_args(10), debug=True)
    W2, m2, v2 = W0.copy(), mb.copy(), vb.copy()
    Wd16, md16, vd16 = fo.adamw_bf16(W2, m2, v2, G, *hp_args(10), debug=True)
    assert np.array_equal(Wd32, Wd16) and np.array_equal(md32, md16) and np.array_equal(vd32, vd16)
    assert np.array_equal(W1, W2)
    assert np.array_equal(m2, fo.f64_to_bf16(md16)) and np.array_equal(v2, fo.f64_to_bf16(vd16))


def test_dgrad_exact_rational_bruteforce_and_adjoint_identity():
    """oracle dgrad (PAPER.md:74 line 1) against exact rational arithmetic on a tiny case, and against the
    adjoint identity <dX, X> = <G, W> that ties it to the pinned wgrad: sum_tq dX[t,q] X[t,q] = sum_pq G[p,q] W[p,q]."""
    from fractions import Fraction
    rng = np.random.default_rng(3)
    T, out, inn = 3, 4, 5
    dY = fo.f64_to_bf16(rng.normal(0, 1, (T, out)))
    W = fo.f64_to_bf16(rng.normal(0, 1, (out, inn)))
    X = fo.f64_to_bf16(rng.normal(0, 1, (T, inn)))
    dX = fo.dgrad(dY, W)
    dYf, Wf = fo.bf16_to_f64(dY), fo.bf16_to_f64(W)
    for t in range(T):
        for q in range(inn):
            exact = sum(Fraction(float(dYf[t, p])) * Fraction(float(Wf[p, q])) for p in range(out))
            assert abs(Fraction(float(dX[t, q])) - exact) <= abs(exact) * Fraction(1, 2 ** 50) + Fraction(1, 2 ** 200)
    G = fo.wgrad(dY, X)
    lhs, rhs = float((dX * fo.bf16_to_f64(X)).sum()), float((G * Wf).sum())
    assert abs(lhs - rhs) <= 1e-12 * (abs(lhs) + abs(rhs) + 1)

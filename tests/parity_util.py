"""Tolerance arithmetic for GPU-vs-oracle parity (BASELINE.json north_star).

e_ij = T * 2^-23 * sum_t |dY_ti||X_tj| bounds the fp32 accumulation error of g.
  m : |dm| <= 1e-4*|m| + (1-b1)*e
  v : |dv| <= 1e-4*v   + (1-b2)*(2|g|e + e^2)
  W : <= 1 bf16 ulp of the oracle's W where |g| > 4e, <= 2*lr (+1 ulp) elsewhere; "1 bf16 ulp"
      carries (reading T1) the fp32 evaluation error of Alg. 1 line 10, 2^-21*(|W_prev| + |W' - W_prev|),
      and the accumulation error of g carried through the update, max |W'(g +- e) - W'(g)| evaluated by the oracle
      in fp64 (`w_prop`) -- the same e the m and v budgets are built on.  Both only matter when decay and update
      cancel W' to ~0 (then an ulp of W' is far below fp32 eps of W); elsewhere they are ~1e-3 of a bf16 ulp
  bf16 moments: + 1 bf16 ulp of the oracle value;  int8: codes +-1, scales rel 1e-3.
All expected values come from oracle/ only.
"""
from __future__ import annotations

import numpy as np
import torch

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import synth

F = np.float32


def hp_tuple(hp):
    return (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])


def bf16_ulp(x: np.ndarray) -> np.ndarray:
    """Spacing of bf16 numbers at |x| (8 significant bits)."""
    a = np.maximum(np.abs(x), 2.0 ** -126)
    return 2.0 ** (np.floor(np.log2(a)) - 7)


def fp32_eval_err(W_prev_bits, Wr):
    """fp32 rounding error of evaluating W' = decay*W - step*ratio (three roundings of terms of size
    |W_prev| and |W' - W_prev|)."""
    if W_prev_bits is None:
        return 0.0
    Wp = fo.bf16_to_f64(W_prev_bits)
    return 2.0 ** -21 * (np.abs(Wp) + np.abs(Wr - Wp))


def to_np(t: torch.Tensor) -> np.ndarray:
    if t.dtype == torch.bfloat16:
        return synth.bf16_bits(t)
    return t.detach().cpu().numpy()


class Tol:
    """Accumulates the state-error budget over chained steps (errors decay with beta)."""

    def __init__(self, shape):
        self.m = np.zeros(shape)
        self.v = np.zeros(shape)
        self.w_ulps = 0

    def step(self, G, E, T, hp):
        b1, b2 = float(F(hp["beta1"])), float(F(hp["beta2"]))
        e = T * 2.0 ** -23 * E
        self.m = b1 * self.m + (1 - b1) * e
        self.v = b2 * self.v + (1 - b2) * (2 * np.abs(G) * e + e * e)
        self.w_ulps += 1
        return e


def w_propagated(kind, W, m, v, G, e, step, hp, scales=None):
    """max |W'(g +- e) - W'(g)| per element, the oracle's own fp64 W' evaluated three times on copies of the state
    BEFORE the step (kind: fp32 | bf16 | int8)."""
    outs = []
    for Gx in (G, G + e, G - e):
        Wc, mc, vc = W.copy(), m.copy(), v.copy()
        if kind == "fp32":
            outs.append(fo.adamw_fp32(Wc, mc, vc, Gx, step, *hp_tuple(hp), debug=True)[0])
        elif kind == "bf16":
            outs.append(fo.adamw_bf16(Wc, mc, vc, Gx, step, *hp_tuple(hp), debug=True)[0])
        else:
            outs.append(fo.adamw_int8(Wc, mc, vc, scales[0].copy(), scales[1].copy(), Gx, step, *hp_tuple(hp), debug=True)[0])
    return np.maximum(np.abs(outs[1] - outs[0]), np.abs(outs[2] - outs[0]))


def _describe(bad, **arrays):
    """First offending element with every quantity that enters its bound (assertion messages)."""
    if not bad.any():
        return ""
    idx = tuple(int(i) for i in np.argwhere(bad)[0])
    return f" first at {idx}: " + ", ".join(f"{k}={np.asarray(a)[idx]!r}" for k, a in arrays.items() if np.ndim(a))


def check_fp(W_gpu, m_gpu, v_gpu, W_or, m_or, v_or, G, e, tol: Tol, hp, moment="fp32", label="", W_prev=None, w_prop=0.0):
    """W_* uint16 bf16 bits; m_*, v_* float32 arrays or uint16 bits (bf16 moments)."""
    lr = float(F(hp["lr"]))
    Wg, Wr = fo.bf16_to_f64(W_gpu), fo.bf16_to_f64(W_or)
    if moment == "bf16":
        mg, mr, vg, vr = (fo.bf16_to_f64(x) for x in (m_gpu, m_or, v_gpu, v_or))
        extra_m, extra_v = bf16_ulp(mr), bf16_ulp(vr)
    else:
        mg, mr, vg, vr = (x.astype(np.float64) for x in (m_gpu, m_or, v_gpu, v_or))
        extra_m = extra_v = 0.0
    dm, dv, dW = np.abs(mg - mr), np.abs(vg - vr), np.abs(Wg - Wr)
    bad_m = dm > 1e-4 * np.abs(mr) + tol.m + extra_m
    bad_v = dv > 1e-4 * np.abs(vr) + tol.v + extra_v
    sure = np.abs(G) > 4 * e
    ulp = bf16_ulp(Wr) + fp32_eval_err(W_prev, Wr) + w_prop
    bad_W = np.where(sure, dW > tol.w_ulps * ulp, dW > 2 * lr * tol.w_ulps + ulp)
    assert not bad_m.any(), f"{label} m: {bad_m.sum()} outside tolerance, worst {dm.max():.3e}" + _describe(bad_m, gpu=mg, oracle=mr, g=G, e=e)
    assert not bad_v.any(), f"{label} v: {bad_v.sum()} outside tolerance, worst {dv.max():.3e}" + _describe(bad_v, gpu=vg, oracle=vr, g=G, e=e)
    assert not bad_W.any(), f"{label} W: {bad_W.sum()} outside tolerance, worst {dW.max():.3e}" + \
        _describe(bad_W, gpu=Wg, oracle=Wr, bound=ulp, g=G, e=e, sure=sure, w_prop=w_prop)
    # the tolerance must not be hiding a systematic error: almost everything is bit-identical
    exact = float((W_gpu == W_or).mean())
    assert exact > 0.99, f"{label} only {exact:.4f} of W bit-identical to the oracle"
    return dict(w_exact=exact, sure=float(sure.mean()), m_rel=float((dm / (np.abs(mr) + 1e-30)).max()))


def check_int8(W_gpu, mq_gpu, vq_gpu, ms_gpu, vs_gpu, W_or, mq_or, vq_or, ms_or, vs_or, G, e, hp, label="", W_prev=None,
               w_prop=0.0):
    lr = float(F(hp["lr"]))
    dq = np.abs(mq_gpu.astype(np.int32) - mq_or.astype(np.int32))
    dvq = np.abs(vq_gpu.astype(np.int32) - vq_or.astype(np.int32))
    assert dq.max() <= 1 and dvq.max() <= 1, f"{label} codes differ by more than 1 ({dq.max()}, {dvq.max()})"
    assert float((dq == 0).mean()) > 0.99 and float((dvq == 0).mean()) > 0.99, f"{label} too many code flips"
    assert np.allclose(ms_gpu, ms_or, rtol=1e-3, atol=0) and np.allclose(vs_gpu, vs_or, rtol=1e-3, atol=0), \
        f"{label} block scales off"
    Wg, Wr = fo.bf16_to_f64(W_gpu), fo.bf16_to_f64(W_or)
    dW = np.abs(Wg - Wr)
    sure = np.abs(G) > 4 * e
    ulp = bf16_ulp(Wr) + fp32_eval_err(W_prev, Wr) + w_prop
    bad_W = np.where(sure, dW > ulp, dW > 2 * lr + ulp)
    assert not bad_W.any(), f"{label} W: {bad_W.sum()} outside tolerance, worst {dW.max():.3e}" + \
        _describe(bad_W, gpu=Wg, oracle=Wr, bound=ulp, g=G, e=e, sure=sure, w_prop=w_prop)
    assert float((W_gpu == W_or).mean()) > 0.99


def sample_rows(out: int, n_ranges: int = 3, width: int = 8, seed: int = 0):
    """Deterministic row ranges spanning the first tile, a middle tile boundary and the last rows."""
    rng = np.random.default_rng(seed + out)
    starts = {0, max(0, out - width)}
    if out > 256:
        starts.add(128 - width // 2)            # straddles the first 128-row tile boundary
    while len(starts) < n_ranges + 2 and out > width:
        starts.add(int(rng.integers(0, out - width)))
    return [(s, min(out, s + width)) for s in sorted(starts)]


def spread_rows(out: int, frac_den: int = 16, width: int = 128):
    """Row ranges covering >= out / frac_den rows, spread uniformly over the whole matrix (every wave of the
    persistent grid, the first and the last rows), with starts that are NOT tile-aligned so that the ranges straddle
    128-row tile and 256-row pair boundaries."""
    n = max(2, -(-out // (frac_den * width)))
    if n * width >= out:
        return [(0, out)]
    starts = [round(k * (out - width) / (n - 1)) for k in range(n)]
    starts = [min(out - width, s + (37 * k) % 64) if 0 < k < n - 1 else s for k, s in enumerate(starts)]
    return [(s, s + width) for s in starts]


def record(kind: str, **kw):
    """Append one line of measured parity statistics (flip rates etc.) to gpurun_out/parity_stats.jsonl; the figures
    quoted in DESIGN.md come from there.  Never read back by any test."""
    import json
    import os
    d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    try:
        os.makedirs(d, exist_ok=True)
        with open(os.path.join(d, "parity_stats.jsonl"), "a") as f:
            f.write(json.dumps(dict(kind=kind, **kw)) + "\n")
    except OSError:
        pass

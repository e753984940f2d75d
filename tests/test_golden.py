"""Golden fixtures (tests/golden/): hand-derived closed-form values pin the oracle; the stored oracle
chain (written by tests/golden/make_golden.py from oracle/ only) detects silent drift of the oracle
and is the expected value of a GPU chained-step test through the C ABI."""
import importlib.util
import os

import numpy as np
import pytest
import torch

from oracle import forge_oracle as fo
from paper_2606_22932_b200 import synth

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
_spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "make_golden.py"))
mg = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(mg)
HP = synth.HP_DEFAULT
HPT = (HP["lr"], HP["beta1"], HP["beta2"], HP["eps"], HP["wd"])


def test_closed_form_step1_hand_values():
    """BASELINE.json north_star closed form, values derived by hand in closed_form_step1.txt."""
    rows = []
    with open(os.path.join(HERE, "closed_form_step1.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 3:
                rows.append((float(line[0]), float(line[1]), int(line[2], 16)))
    assert len(rows) == 5
    for w, g, expect in rows:
        W = synth.bf16_bits(torch.tensor([[w]], dtype=torch.bfloat16)).copy()
        assert fo.bf16_to_f64(W)[0, 0] == w                      # the fixture's W is bf16-exact
        m = np.zeros((1, 1), np.float32); v = np.zeros((1, 1), np.float32)
        fo.adamw_fp32(W, m, v, np.array([[g]], np.float64), 1, *HPT)
        assert int(W[0, 0]) == expect, (w, g, hex(int(W[0, 0])), hex(expect))
        assert m[0, 0] == np.float32((1 - np.float64(np.float32(0.9))) * g)
        assert v[0, 0] == np.float32((1 - np.float64(np.float32(0.999))) * g * g)


def test_stored_chain_is_what_the_oracle_computes_today():
    stored, now = mg.load(), mg.run()
    assert set(stored) == set(now)
    for k in stored:
        assert np.array_equal(stored[k], now[k]), f"oracle drifted on {k}: regenerate only with a cited reason"


@pytest.mark.gpu
@pytest.mark.parametrize("moment", ["fp32", "bf16", "int8"])
def test_gpu_chain_against_stored_oracle_values(moment):
    from paper_2606_22932_b200 import binding as fb
    import parity_util as pu
    g = mg.load()
    dev = "cuda"
    W = synth.bits_to_bf16(mg.initial()).to(dev)
    z = torch.zeros(mg.OUT, mg.IN, device=dev)
    kw = {}
    if moment == "fp32":
        m, v = z.clone(), z.clone()
    elif moment == "bf16":
        m, v = z.to(torch.bfloat16), z.to(torch.bfloat16)
    else:
        m, v = z.to(torch.int8), z.to(torch.uint8)
        kw = dict(m_scale=torch.zeros(mg.OUT, 1, device=dev), v_scale=torch.zeros(mg.OUT, 1, device=dev))
    for step in range(1, mg.STEPS + 1):
        X, dY = mg.inputs(step)
        fb.forge_wgrad_adamw(synth.bits_to_bf16(X).to(dev), synth.bits_to_bf16(dY).to(dev), W, m, v, step, *HPT, **kw)
    torch.cuda.synchronize()
    Wg, Wr = fo.bf16_to_f64(synth.bf16_bits(W)), fo.bf16_to_f64(g[f"{moment}_W"])
    # three chained steps: each step's W' is within 1 bf16 ulp, or 2*lr where the sign of g is not determined
    # (north_star); the element-wise |g| > 4e split is exercised in test_gpu_parity.py, here the loose union
    # bound plus "almost all bit-identical" guards against drift of either side
    assert np.all(np.abs(Wg - Wr) <= 3 * pu.bf16_ulp(Wr) + 3 * 2 * HP["lr"])
    assert float((synth.bf16_bits(W) == g[f"{moment}_W"]).mean()) > 0.98
    if moment == "fp32":
        assert np.allclose(m.cpu().numpy(), g["fp32_m"], rtol=2e-4, atol=1e-9)
        assert np.allclose(v.cpu().numpy(), g["fp32_v"], rtol=2e-4, atol=1e-12)
    elif moment == "int8":
        assert np.abs(m.cpu().numpy().astype(int) - g["int8_m"].astype(int)).max() <= 1
        assert np.abs(v.cpu().numpy().astype(int) - g["int8_v"].astype(int)).max() <= 1
        assert np.allclose(kw["m_scale"].cpu().numpy(), g["int8_m_scale"], rtol=1e-3)
        assert np.allclose(kw["v_scale"].cpu().numpy(), g["int8_v_scale"], rtol=1e-3)

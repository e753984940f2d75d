#!/usr/bin/env python
"""Writes tests/golden/chain3_small.txt: a scaled-down BASELINE.json configs[0] (three chained steps,
fresh inputs per step) evaluated by the ORACLE ONLY, for fp32, bf16 and int8 moments.  Nothing here
touches the CUDA path.  Re-run after a justified change to the oracle's arithmetic:

    python tests/golden/make_golden.py

Layout of the text file: `key shape dtype hex-bytes` per line (little endian, C order).
Inputs are not stored: they are regenerated from the seeds by paper_2606_22932_b200/synth.py
(random draws and dtype casts only)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import forge_oracle as fo                     # noqa: E402
from paper_2606_22932_b200 import synth                   # noqa: E402

OUT, IN, T, STEPS, SEED = 8, 256, 40, 3, 424242
HP = synth.HP_DEFAULT
PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "chain3_small.txt")


def inputs(step):
    p = synth.make_problem("g", T, OUT, IN, SEED + step, sigma_dy=1e-2)
    return synth.bf16_bits(p.X), synth.bf16_bits(p.dY)


def initial():
    p = synth.make_problem("g", T, OUT, IN, SEED, zero_state=True)
    return synth.bf16_bits(p.W).copy()


def run():
    hp = (HP["lr"], HP["beta1"], HP["beta2"], HP["eps"], HP["wd"])
    res = {}
    W = initial(); m = np.zeros((OUT, IN), np.float32); v = np.zeros((OUT, IN), np.float32)
    Wb = initial(); mb = np.zeros((OUT, IN), np.uint16); vb = np.zeros((OUT, IN), np.uint16)
    Wq = initial(); mq, ms, vq, vs = fo.quantize(np.zeros((OUT, IN)), np.zeros((OUT, IN)))
    for step in range(1, STEPS + 1):
        X, dY = inputs(step)
        G = fo.wgrad(dY, X)
        fo.adamw_fp32(W, m, v, G, step, *hp)
        fo.adamw_bf16(Wb, mb, vb, G, step, *hp)
        fo.adamw_int8(Wq, mq, vq, ms, vs, G, step, *hp)
    res.update(fp32_W=W, fp32_m=m, fp32_v=v, bf16_W=Wb, bf16_m=mb, bf16_v=vb,
               int8_W=Wq, int8_m=mq, int8_v=vq, int8_m_scale=ms, int8_v_scale=vs)
    return res


def load(path=PATH):
    out = {}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            key, shape, dtype, hx = line.split()
            out[key] = np.frombuffer(bytes.fromhex(hx), dtype=dtype).reshape([int(s) for s in shape.split("x")]).copy()
    return out


if __name__ == "__main__":
    res = run()
    with open(PATH, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; OUT=%d IN=%d T=%d steps=%d seed=%d\n"
                % (OUT, IN, T, STEPS, SEED))
        f.write("# method: PAPER.md:72-74 Algorithm 1; int8 per PAPER.md:316 with DESIGN.md readings S4-S7\n")
        for k, a in res.items():
            a = np.ascontiguousarray(a)
            f.write("%s %s %s %s\n" % (k, "x".join(map(str, a.shape)), a.dtype.str, a.tobytes().hex()))
    print("wrote", PATH, os.path.getsize(PATH), "bytes")

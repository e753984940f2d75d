"""Seeded synthetic inputs shaped like the paper's Llama-3.1-8B workloads.

This module serves BOTH the CUDA path's callers (tests, bench.py) and the oracle's callers; it
holds none of the method's arithmetic -- only random draws and torch's own dtype casts.  The
recipe follows BASELINE.json `configs` (second argument of N(0, x) read as the standard
deviation, reading S12).  The paper's timing and memory cells are random-init and
"shape-deterministic"; these tensors stand in for its datasets and
checkpoints, which are not available here.
"""
from __future__ import annotations

from dataclasses import dataclass

import torch

BASE_SEED = 20260622

# (name, out, in) of one Llama-3.1-8B decoder layer's seven projections (BASELINE.json cfg 1).
LLAMA8B_LAYER = (
    ("q", 4096, 4096), ("k", 1024, 4096), ("v", 1024, 4096), ("o", 4096, 4096),
    ("gate", 14336, 4096), ("up", 14336, 4096), ("down", 4096, 14336),
)
LLAMA8B_LM_HEAD = ("lm_head", 128256, 4096)
# which projections read the same activation X (q/k/v share one, gate/up share one)
X_GROUP = {"q": "attn_in", "k": "attn_in", "v": "attn_in", "o": "o_in",
           "gate": "mlp_in", "up": "mlp_in", "down": "down_in", "lm_head": "head_in"}

HP_DEFAULT = dict(lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.1)


@dataclass
class Problem:
    """One linear layer's tensors.  bf16 tensors are torch.bfloat16; moments fp32 seeds."""
    name: str
    T: int
    out: int
    inn: int
    X: torch.Tensor      # [T, in]  bf16
    dY: torch.Tensor     # [T, out] bf16
    W: torch.Tensor      # [out, in] bf16
    m: torch.Tensor      # [out, in] fp32 seed
    v: torch.Tensor      # [out, in] fp32 seed (>= 0)


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def randn_bf16(shape, sigma: float, seed: int, device="cpu") -> torch.Tensor:
    x = torch.randn(shape, generator=_gen(seed, device), dtype=torch.float32, device=device)
    return (x * sigma).to(torch.bfloat16)


def randn_f32(shape, sigma: float, seed: int, device="cpu", absval: bool = False) -> torch.Tensor:
    x = torch.randn(shape, generator=_gen(seed, device), dtype=torch.float32, device=device) * sigma
    return x.abs() if absval else x


def make_problem(name: str, T: int, out: int, inn: int, seed: int, *, sigma_x=1.0, sigma_dy=1e-3,
                 sigma_w=0.02, sigma_m=1e-4, sigma_v=1e-6, zero_state=False, device="cpu",
                 X: torch.Tensor | None = None) -> Problem:
    """Config-1 distributions by default; `zero_state` gives config 0's m = v = 0."""
    if X is None:
        X = randn_bf16((T, inn), sigma_x, seed * 16 + 1, device)
    dY = randn_bf16((T, out), sigma_dy, seed * 16 + 2, device)
    W = randn_bf16((out, inn), sigma_w, seed * 16 + 3, device)
    if zero_state:
        m = torch.zeros((out, inn), dtype=torch.float32, device=device)
        v = torch.zeros((out, inn), dtype=torch.float32, device=device)
    else:
        m = randn_f32((out, inn), sigma_m, seed * 16 + 4, device)
        v = randn_f32((out, inn), sigma_v, seed * 16 + 5, device, absval=True)
    return Problem(name, T, out, inn, X, dY, W, m, v)


def make_layer(T: int, seed: int, shapes=LLAMA8B_LAYER, device="cpu", **kw) -> list[Problem]:
    """All projections of one decoder layer; projections in one X_GROUP share the same X."""
    xs: dict[tuple[str, int], torch.Tensor] = {}
    probs = []
    for i, (name, out, inn) in enumerate(shapes):
        key = (X_GROUP.get(name, name), inn)
        if key not in xs:
            xs[key] = randn_bf16((T, inn), kw.get("sigma_x", 1.0), seed * 1000 + 100 + len(xs), device)
        probs.append(make_problem(name, T, out, inn, seed * 1000 + i, X=xs[key], device=device, **kw))
    return probs


def random_int8_state(out: int, inn: int, seed: int, device="cpu", block: int = 256):
    """Synthetic int8 blockwise optimizer state drawn DIRECTLY as codes and scales (no quantiser arithmetic: the timed
    path is data-independent, and the parity tests seed theirs with the oracle's quantiser instead): m codes
    ~ round(N(0, 40)) clipped to [-127, 127], v codes uniform in [1, 255], block scales of the cfg-1 magnitudes
    (absmax of 256 draws of N(0, 1e-4) resp. |N(0, 1e-6)| is about 3 sigma).  Returns (m, v, m_scale, v_scale)."""
    g = _gen(seed, device)
    m = (torch.randn((out, inn), generator=g, dtype=torch.float32, device=device) * 40.0).round_().clamp_(-127, 127).to(torch.int8)
    v = torch.randint(1, 256, (out, inn), generator=g, dtype=torch.int32, device=device).to(torch.uint8)
    nb = inn // block
    ms = (3e-4 + 1e-4 * torch.rand((out, nb), generator=g, dtype=torch.float32, device=device)).contiguous()
    vs = (3e-6 + 1e-6 * torch.rand((out, nb), generator=g, dtype=torch.float32, device=device)).contiguous()
    return m, v, ms, vs


def random_fp8_state(out: int, inn: int, seed: int, device="cpu"):
    """Synthetic e4m3 optimizer state drawn directly as codes (never the NaN code 0x7F / 0xFF) with one {scale, amax
    out} pair per tensor.  Returns (m, v, m_scale, v_scale)."""
    g = _gen(seed, device)
    mag = torch.randint(0, 0x7F, (out, inn), generator=g, dtype=torch.int32, device=device)
    sign = torch.randint(0, 2, (out, inn), generator=g, dtype=torch.int32, device=device) * 0x80
    m = (mag | sign).to(torch.uint8)
    v = torch.randint(1, 0x7F, (out, inn), generator=g, dtype=torch.int32, device=device).to(torch.uint8)
    ms = torch.tensor([3e-4 / 448.0, 0.0], dtype=torch.float32, device=device)
    vs = torch.tensor([3e-6 / 448.0, 0.0], dtype=torch.float32, device=device)
    return m, v, ms, vs


def config0_step_inputs(step: int, device="cpu"):
    """BASELINE.json cfg 0: fresh X[128,256] ~N(0,1), dY[128,384] ~N(0,1e-2) per step."""
    s = BASE_SEED + 7919 * step
    return randn_bf16((128, 256), 1.0, s * 16 + 1, device), randn_bf16((128, 384), 1e-2, s * 16 + 2, device)


def config0_weight(device="cpu") -> torch.Tensor:
    return randn_bf16((384, 256), 0.02, BASE_SEED * 16 + 3, device)


def bf16_bits(t: torch.Tensor):
    """torch.bfloat16 tensor -> numpy uint16 bit patterns (a view change, no arithmetic)."""
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view("uint16")


def bits_to_bf16(a) -> torch.Tensor:
    import numpy as np
    return torch.from_numpy(np.ascontiguousarray(a).view("int16")).view(torch.bfloat16)

"""BASELINE.json configs[4]: the full Llama-3.1-8B linear stack resident on one B200 -- 32 decoder
layers of 7 projections plus lm_head W[128256,4096], bf16 W + fp32 m/v (75.05 GB of state) -- and one
optimizer step taken layer by layer in REVERSE order, the order the backward pass visits the layers
(PAPER.md:25, 27, 64).  Only allocation, seeding and the order of the C-ABI calls live here; every
arithmetic step runs in the CUDA library.

Two arms:
  fused    : one forge_wgrad_adamw_grouped call per layer (lm_head first); no dW exists anywhere.
  dw_pool  : the conventional schedule the paper compares against: every layer's
             gradient is MATERIALISED (cuBLAS dW = dY^T X into an fp32 pool that lives until the
             optimizer phase, 4 B / parameter = 30 GB), then one elementwise AdamW pass over the pool.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import torch

from . import binding as fb
from . import synth

N_LAYERS = 32


@dataclass
class Stack:
    layers: list = field(default_factory=list)     # list (len 33) of lists of problem dicts; last = [lm_head]
    arrays: list = field(default_factory=list)     # matching forge_problem_t arrays
    params: int = 0
    state_bytes: int = 0
    input_bytes: int = 0


def build_stack(device, tokens: int = 512, n_layers: int = N_LAYERS, seed: int = synth.BASE_SEED + 4,
                lm_head: bool = True, share_inputs: bool = False) -> Stack:
    """Seeded cfg-1 distributions for every layer (synth.make_layer on the device).  With
    `share_inputs` all layers read layer 0's X/dY tensors (saves 2.6 GB; shapes are identical)."""
    st = Stack()
    shapes_list = [synth.LLAMA8B_LAYER] * n_layers + ([(synth.LLAMA8B_LM_HEAD,)] if lm_head else [])
    first = None
    for li, shapes in enumerate(shapes_list):
        probs = synth.make_layer(tokens, seed * 100 + li, shapes=shapes, device=device)
        layer = []
        for pi, p in enumerate(probs):
            d = dict(name=f"L{li}.{p.name}", X=p.X, dY=p.dY, W=p.W, m=p.m, v=p.v)
            if share_inputs and first is not None and len(shapes) == len(synth.LLAMA8B_LAYER):
                d["X"], d["dY"] = first[pi]["X"], first[pi]["dY"]
            layer.append(d)
            st.params += p.out * p.inn
        if first is None:
            first = layer
        st.layers.append(layer)
        st.arrays.append(fb.make_problem_array(layer))
    st.state_bytes = st.params * 10
    seen = set()
    for layer in st.layers:
        for d in layer:
            for k in ("X", "dY"):
                if d[k].data_ptr() not in seen:
                    seen.add(d[k].data_ptr())
                    st.input_bytes += d[k].numel() * 2
    return st


def step_fused(st: Stack, step: int, hp: dict, stream=None) -> int:
    """One optimizer step, deepest layer first: lm_head, then layers 31 .. 0.  Returns launches."""
    n0 = fb.forge_launch_count()
    for layer, arr in zip(reversed(st.layers), reversed(st.arrays)):
        fb.forge_wgrad_adamw_grouped(layer, step, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"],
                                     fb.FP32, stream=stream, _arr=arr)
    return fb.forge_launch_count() - n0


def alloc_dw_pool(st: Stack, device):
    """The materialised fp32 gradient pool of the conventional schedule: one tensor per weight."""
    return [[torch.empty(d["W"].shape, dtype=torch.float32, device=device) for d in layer] for layer in st.layers]


def step_dw_pool(st: Stack, pool, step: int, hp: dict):
    """Backward phase: cuBLAS dW for every layer in reverse order into the pool; optimizer phase:
    the library's elementwise AdamW kernel over every pooled gradient (test/bench-only symbol)."""
    for layer, grads in zip(reversed(st.layers), reversed(pool)):
        for d, G in zip(layer, grads):
            torch.mm(d["dY"].t(), d["X"], out_dtype=torch.float32, out=G)
    for layer, grads in zip(reversed(st.layers), reversed(pool)):
        for d, G in zip(layer, grads):
            fb.forge_adamw_from_g(G, d["W"], d["m"], d["v"], step, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])

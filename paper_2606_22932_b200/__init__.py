"""forge-b200: FORGE's fused weight-gradient + AdamW hot path (arxiv/paper_2606_22932) for sm_100a.

The compute lives in ``csrc/`` behind the C ABI declared in ``include/forge.h``; ``binding`` is a
thin ctypes layer with the same names.  Nothing here falls back to a CPU or library path: if the
CUDA library is missing, ``binding`` raises.
"""
__all__ = ["binding", "synth", "build"]

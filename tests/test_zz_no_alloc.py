"""forge_wgrad_adamw_host_noalloc (include/forge.h): the host-buffer entry whose device staging is the library's
static 32 MiB __device__ array -- for callers that may not call cudaMalloc.  Checked against the existing paths
(forge_wgrad_adamw_host, which allocates its staging, and the device-resident forge_wgrad_adamw) with the bar the
other host-entry test uses: bit-identical W, m, v (and int8 codes / scales).

Kept in a file of its own that pytest collects last (the suite runs with `pytest -x`).  It depends on no other test:
each call overwrites every region of the shared array it reads, so the order of tests cannot matter.
"""
import pytest
import torch

from paper_2606_22932_b200 import binding as fb
from paper_2606_22932_b200 import synth

HP = synth.HP_DEFAULT
TOO_LARGE = fb.STATUS_NAMES.index("FORGE_ERR_TOO_LARGE")


def _host_problem(T, out, inn, seed, moments):
    """One seeded problem in host memory: operands + state in the layout of the requested moment dtype."""
    p = synth.make_problem("x", T, out, inn, seed=seed)
    h = dict(X=p.X.clone(), dY=p.dY.clone(), W=p.W.clone())
    if moments == "fp32":
        h["m"], h["v"] = p.m.clone(), p.v.clone()
    elif moments == "bf16":
        h["m"], h["v"] = p.m.to(torch.bfloat16), p.v.to(torch.bfloat16)
    else:
        h["m"], h["v"], h["m_scale"], h["v_scale"] = synth.random_int8_state(out, inn, seed + 1000)
    return h


def _clone(h):
    return {k: t.clone() for k, t in h.items()}


def _state_keys(h):
    return [k for k in ("W", "m", "v", "m_scale", "v_scale") if k in h]


def _call(fn, h, step):
    fn(h["X"], h["dY"], h["W"], h["m"], h["v"], step, m_scale=h.get("m_scale"), v_scale=h.get("v_scale"), **HP)


def test_too_large_is_rejected_before_any_cuda_call():
    """CPU: fake, never dereferenced pointers.  2048 x 2048 with fp32 moments stages 44 MiB > the 32 MiB array."""
    L = fb.lib()
    ptrs = [0x10000000 * k for k in range(1, 6)]
    hp = (1, 1e-3, 0.9, 0.999, 1e-8, 0.1)
    assert L.forge_wgrad_adamw_host_noalloc(*ptrs, None, None, 512, 2048, 2048, *hp, fb.FP32) == TOO_LARGE
    assert L.forge_wgrad_adamw_host_noalloc(*ptrs, None, None, 0, 256, 256, *hp, fb.FP32) == 2      # BAD_SHAPE first
    assert L.forge_wgrad_adamw_host_noalloc(None, *ptrs[1:], None, None, 128, 256, 256, *hp, fb.FP32) == 1
    assert fb.forge_status_string(TOO_LARGE) == "FORGE_ERR_TOO_LARGE"
    assert fb.NOALLOC_SCRATCH_BYTES == 32 << 20


@pytest.mark.gpu
def test_no_alloc_entry_matches_the_existing_paths_on_calls_in_a_row():
    """Three calls back to back through the SAME static array, each a different shape and moment dtype (so each one
    lands on the previous call's bytes at different offsets), then the first one again: every result bit-identical to
    forge_wgrad_adamw_host, and the first also to the device-resident forge_wgrad_adamw."""
    cases = [(128, 256, 512, 31, "fp32", 6),      # several tiles
             (96, 384, 768, 32, "int8", 3),       # ragged token count, codes + block scales, smaller footprint
             (512, 1024, 1536, 33, "bf16", 9),    # 11.5 MiB staged: multi-wave, well past the earlier footprints
             (128, 256, 512, 31, "fp32", 6)]      # the first again, now over bytes two other calls left behind
    launches0 = fb.forge_launch_count()
    for T, out, inn, seed, moments, step in cases:
        h0 = _host_problem(T, out, inn, seed, moments)
        ref, new = _clone(h0), _clone(h0)
        _call(fb.forge_wgrad_adamw_host, ref, step)
        _call(fb.forge_wgrad_adamw_host_noalloc, new, step)
        for k in _state_keys(h0):
            assert torch.equal(ref[k], new[k]), f"{moments} {out}x{inn}: {k} differs from forge_wgrad_adamw_host"
        assert not torch.equal(new["W"], h0["W"]) and not torch.equal(new["m"], h0["m"])    # the step did run
        assert torch.equal(new["X"], h0["X"]) and torch.equal(new["dY"], h0["dY"])          # operands are read-only
    assert fb.forge_launch_count() - launches0 == 2 * len(cases)                            # one fused launch per call

    # two calls in a row on ONE state (steps 1 and 2), against the device-resident path doing the same two steps
    h0 = _host_problem(128, 256, 512, 41, "fp32")
    new = _clone(h0)
    d = {k: t.cuda() for k, t in h0.items()}
    for step in (1, 2):
        _call(fb.forge_wgrad_adamw_host_noalloc, new, step)
        fb.forge_wgrad_adamw(d["X"], d["dY"], d["W"], d["m"], d["v"], step, **HP)
    torch.cuda.synchronize()
    for k in ("W", "m", "v"):
        assert torch.equal(d[k].cpu(), new[k]), f"{k} differs from forge_wgrad_adamw after two steps"


@pytest.mark.gpu
def test_no_alloc_entry_rejects_what_does_not_fit_and_touches_nothing():
    h0 = _host_problem(64, 2048, 2048, 51, "fp32")          # 40.5 MiB of staging
    new = _clone(h0)
    st = fb.forge_wgrad_adamw_host_noalloc(new["X"], new["dY"], new["W"], new["m"], new["v"], 1, check=False, **HP)
    assert st == TOO_LARGE
    with pytest.raises(fb.ForgeError, match="FORGE_ERR_TOO_LARGE"):
        _call(fb.forge_wgrad_adamw_host_noalloc, new, 1)
    for k in _state_keys(h0):
        assert torch.equal(new[k], h0[k])
    # the same shape fits with int8 moments (2 + 2 * 1.016 bytes per element): the limit is on staged bytes, not on shape
    h1 = _host_problem(64, 2048, 2048, 52, "int8")
    ref, new = _clone(h1), _clone(h1)
    _call(fb.forge_wgrad_adamw_host, ref, 2)
    _call(fb.forge_wgrad_adamw_host_noalloc, new, 2)
    for k in _state_keys(h1):
        assert torch.equal(ref[k], new[k])

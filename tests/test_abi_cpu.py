"""Host-side checks of the C ABI that need no GPU: the library loads, exports every symbol that
include/forge.h declares, and rejects bad arguments before touching CUDA."""
import ctypes
import os
import re

import pytest

from paper_2606_22932_b200 import binding as fb
from paper_2606_22932_b200 import build as cuda_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HP = (10, 1e-3, 0.9, 0.999, 1e-8, 0.1)


@pytest.fixture(scope="module")
def lib():
    cuda_build.build()
    return fb.lib()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "forge.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(forge_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert "forge_wgrad_adamw" in names and "forge_wgrad_adamw_grouped" in names and len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/forge.h but not exported"
    assert sorted(fb.EXPORTS) == names


def test_version_strings_workspace(lib):
    assert fb.forge_version() == 100
    assert fb.forge_workspace_bytes() == 0          # no O(out*in) term: dW is never allocated
    assert [fb.forge_status_string(i) for i in range(len(fb.STATUS_NAMES))] == fb.STATUS_NAMES
    assert fb.forge_status_string(99) == "FORGE_ERR_UNKNOWN"


def test_struct_layout_matches_header():
    # 7 pointers + 3 int32 padded to 8 + the two operand pitches (ldx, lddy)
    assert ctypes.sizeof(fb.forge_problem_t) == 7 * 8 + 16 + 16
    assert fb.forge_problem_t.T.offset == 56 and fb.forge_problem_t.in_.offset == 64
    assert fb.forge_problem_t.ldx.offset == 72 and fb.forge_problem_t.lddy.offset == 80


# fake device pointers, far enough apart that no tensor of a call overlaps another
PX, PDY, PW, PM, PV, PMS, PVS = (0x10000000 * k for k in range(1, 8))


def _call(lib, X=PX, dY=PDY, W=PW, m=PM, v=PV, ms=None, vs=None, T=128, out=384, inn=256,
          hp=HP, mdt=0):
    return lib.forge_wgrad_adamw(X, dY, W, m, v, ms, vs, T, out, inn, *hp, mdt, None)


def test_argument_validation_happens_before_any_cuda_call(lib):
    """Fake (never dereferenced) pointers: every one of these must be rejected on a box with no GPU."""
    NULL_PTR, BAD_SHAPE, ALIGN, BAD_HP, BAD_DT = 1, 2, 3, 4, 5
    assert _call(lib, X=None) == NULL_PTR and _call(lib, dY=None) == NULL_PTR
    assert _call(lib, W=None) == NULL_PTR and _call(lib, m=None) == NULL_PTR and _call(lib, v=None) == NULL_PTR
    assert _call(lib, T=0) == BAD_SHAPE                      # decay-only case rejected (Remark 1)
    assert _call(lib, out=0) == BAD_SHAPE and _call(lib, out=100) == BAD_SHAPE and _call(lib, inn=12) == BAD_SHAPE
    assert _call(lib, W=PW + 8) == ALIGN and _call(lib, X=PX + 2) == ALIGN and _call(lib, m=PM + 4) == ALIGN
    assert _call(lib, hp=(0, 1e-3, 0.9, 0.999, 1e-8, 0.1)) == BAD_HP       # step is 1-based
    assert _call(lib, hp=(1, -1.0, 0.9, 0.999, 1e-8, 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 1.0, 0.999, 1e-8, 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 0.9, -0.1, 1e-8, 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 0.9, 0.999, float("nan"), 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 0.9, 0.999, 1e-8, -1.0)) == BAD_HP
    assert _call(lib, mdt=4) == BAD_DT and _call(lib, mdt=-1) == BAD_DT
    assert _call(lib, mdt=3) == NULL_PTR                      # FP8 needs its scale / amax pairs
    assert _call(lib, mdt=3, ms=PMS, vs=PVS, inn=264) == BAD_SHAPE   # in % 16 for 1-byte codes
    assert _call(lib, mdt=0, ms=PMS, vs=PVS) == BAD_DT  # scales only with INT8
    assert _call(lib, mdt=2) == NULL_PTR                      # INT8 needs scales
    assert _call(lib, mdt=2, ms=PMS, vs=PVS, inn=384) == BAD_SHAPE   # in % 256
    # grouped: null array, empty group, one bad member rejects the whole group
    assert lib.forge_wgrad_adamw_grouped(None, 1, *HP, 0, None) == NULL_PTR
    arr = (fb.forge_problem_t * 2)()
    for k, a in enumerate(arr):
        a.X, a.dY, a.T, a.out, a.in_ = PX, PDY, 128, 384, 256           # the operands may be shared
        a.W, a.m, a.v = PW + k * 0x1000000, PM + k * 0x1000000, PV + k * 0x1000000
    assert lib.forge_wgrad_adamw_grouped(arr, 0, *HP, 0, None) == BAD_SHAPE
    arr[1].out = 7
    assert lib.forge_wgrad_adamw_grouped(arr, 2, *HP, 0, None) == BAD_SHAPE
    # operand pitches: 0 = dense; otherwise >= the row length and a multiple of 8 elements
    arr[1].out = 384
    for ldx, lddy in ((255, 0), (260, 0), (0, 380), (0, 388)):
        arr[1].ldx, arr[1].lddy = ldx, lddy
        assert lib.forge_wgrad_adamw_grouped(arr, 2, *HP, 0, None) == BAD_SHAPE
    arr[1].ldx, arr[1].lddy = 512, 1152                       # valid strided views are refused by the host-buffer entry only
    assert lib.forge_wgrad_adamw_grouped_host(arr, 2, *HP, 0) == BAD_SHAPE
    arr[1].ldx, arr[1].lddy = 0, 0
    # test-only twins validate too
    assert lib.forge_wgrad_store_g(None, PDY, PW, 128, 384, 256, None) == NULL_PTR
    assert lib.forge_adamw_from_g(None, PW, PM, PV, None, None, 384, 256, *HP, 0, None) == NULL_PTR
    assert lib.forge_wgrad_adamw_host(PX, PDY, PW, PM, PV, None, None, 0, 384, 256, *HP, 0) == BAD_SHAPE
    # the widened entries validate the operand pitches too (they used to surface as a tensor-map failure)
    opt = fb.forge_opt_desc_t(family=1, nesterov=0, step=1, lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.0, momentum=0.0)
    one = (fb.forge_problem_t * 1)()
    one[0].X, one[0].dY, one[0].W, one[0].T, one[0].out, one[0].in_, one[0].ldx = PX, PDY, PW, 128, 384, 256, 100
    assert lib.forge_wgrad_step_grouped(one, 1, ctypes.byref(opt), 0, None) == BAD_SHAPE
    one[0].W, one[0].m = None, PM
    assert lib.forge_wgrad_accumulate_grouped(one, 1, 0.5, 0, None) == BAD_SHAPE
    assert lib.forge_wgrad_store_g_grouped(one, 1, None) == BAD_SHAPE


def test_overlapping_state_is_rejected_before_any_cuda_call(lib):
    """forge.h "Aliasing (enforced)": an updated tensor may not overlap any other tensor of the call."""
    BAD_SHAPE = 2
    n = 384 * 256
    # inside one problem: m starts inside W; v == m; W inside X; scales on top of codes
    assert _call(lib, m=PW + n) == BAD_SHAPE          # W is 2n bytes long
    assert _call(lib, v=PM) == BAD_SHAPE
    assert _call(lib, W=PX + 64) == BAD_SHAPE
    assert _call(lib, mdt=2, ms=PM + 256, vs=PVS) == BAD_SHAPE
    # across the problems of a group: the same W twice; a W that ends inside the next problem's m
    arr = (fb.forge_problem_t * 3)()
    for k, a in enumerate(arr):
        a.X, a.dY, a.T, a.out, a.in_ = PX, PDY, 128, 384, 256
        a.W, a.m, a.v = PW + k * 0x1000000, PM + k * 0x1000000, PV + k * 0x1000000
    arr[2].W = arr[0].W
    assert lib.forge_wgrad_adamw_grouped(arr, 3, *HP, 0, None) == BAD_SHAPE
    arr[2].W = arr[1].m - 2 * n + 16
    assert lib.forge_wgrad_adamw_grouped(arr, 3, *HP, 0, None) == BAD_SHAPE
    # adjacent (touching, not overlapping) tensors are fine: the call gets as far as the device query
    arr[2].W = arr[1].m - 2 * n
    assert lib.forge_wgrad_adamw_grouped(arr, 3, *HP, 0, None) != BAD_SHAPE
    # layer backward: dX may not overlap the state
    dx = (ctypes.c_void_p * 3)(0x70000000, 0x71000000, arr[0].v + 32)
    assert lib.forge_layer_backward_grouped(arr, dx, 3, *HP, 0, None) == BAD_SHAPE


def test_product_library_has_no_profiling_switches():
    """FORGE_ABLATE / FORGE_GRID / FORGE_CFG are compiled only into the -DFORGE_PROFILING build; the product library
    links no GEMM library (the dgrad is hand-written)."""
    blob = open(cuda_build.build(), "rb").read()
    for name in (b"FORGE_ABLATE", b"FORGE_GRID", b"FORGE_CFG", b"FORGE_POWER_STATE", b"FORGE_HOST_SLICE_MB", b"cublas"):
        assert name not in blob, name
    prof = open(cuda_build.build(profiling=True), "rb").read()
    assert b"FORGE_ABLATE" in prof and b"FORGE_GRID" in prof and b"FORGE_CFG" in prof


def test_product_package_does_not_import_the_oracle():
    """The product path must never route through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_22932_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("forge_oracle", "oracle") or f == "synth.py", f
    oracle_src = open(os.path.join(ROOT, "oracle", "forge_oracle.py")).read() + \
        open(os.path.join(ROOT, "oracle", "forge_oracle.c")).read()
    assert "import paper_2606_22932_b200" not in oracle_src and "from paper_2606_22932_b200" not in oracle_src
    assert "#include \"../" not in oracle_src and "forge.h" not in oracle_src

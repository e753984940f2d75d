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
    assert [fb.forge_status_string(i) for i in range(8)] == fb.STATUS_NAMES
    assert fb.forge_status_string(99) == "FORGE_ERR_UNKNOWN"


def test_struct_layout_matches_header():
    # 7 pointers + 3 int32 padded to 8 + the two operand pitches (ldx, lddy)
    assert ctypes.sizeof(fb.forge_problem_t) == 7 * 8 + 16 + 16
    assert fb.forge_problem_t.T.offset == 56 and fb.forge_problem_t.in_.offset == 64
    assert fb.forge_problem_t.ldx.offset == 72 and fb.forge_problem_t.lddy.offset == 80


def _call(lib, X=0x1000, dY=0x2000, W=0x3000, m=0x4000, v=0x5000, ms=None, vs=None, T=128, out=384, inn=256,
          hp=HP, mdt=0):
    return lib.forge_wgrad_adamw(X, dY, W, m, v, ms, vs, T, out, inn, *hp, mdt, None)


def test_argument_validation_happens_before_any_cuda_call(lib):
    """Fake (never dereferenced) pointers: every one of these must be rejected on a box with no GPU."""
    NULL_PTR, BAD_SHAPE, ALIGN, BAD_HP, BAD_DT = 1, 2, 3, 4, 5
    assert _call(lib, X=None) == NULL_PTR and _call(lib, dY=None) == NULL_PTR
    assert _call(lib, W=None) == NULL_PTR and _call(lib, m=None) == NULL_PTR and _call(lib, v=None) == NULL_PTR
    assert _call(lib, T=0) == BAD_SHAPE                      # decay-only case rejected (Remark 1)
    assert _call(lib, out=0) == BAD_SHAPE and _call(lib, out=100) == BAD_SHAPE and _call(lib, inn=12) == BAD_SHAPE
    assert _call(lib, W=0x3008) == ALIGN and _call(lib, X=0x1002) == ALIGN and _call(lib, m=0x4004) == ALIGN
    assert _call(lib, hp=(0, 1e-3, 0.9, 0.999, 1e-8, 0.1)) == BAD_HP       # step is 1-based
    assert _call(lib, hp=(1, -1.0, 0.9, 0.999, 1e-8, 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 1.0, 0.999, 1e-8, 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 0.9, -0.1, 1e-8, 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 0.9, 0.999, float("nan"), 0.1)) == BAD_HP
    assert _call(lib, hp=(1, 1e-3, 0.9, 0.999, 1e-8, -1.0)) == BAD_HP
    assert _call(lib, mdt=4) == BAD_DT and _call(lib, mdt=-1) == BAD_DT
    assert _call(lib, mdt=3) == NULL_PTR                      # FP8 needs its scale / amax pairs
    assert _call(lib, mdt=3, ms=0x6000, vs=0x7000, inn=264) == BAD_SHAPE   # in % 16 for 1-byte codes
    assert _call(lib, mdt=0, ms=0x6000, vs=0x7000) == BAD_DT  # scales only with INT8
    assert _call(lib, mdt=2) == NULL_PTR                      # INT8 needs scales
    assert _call(lib, mdt=2, ms=0x6000, vs=0x7000, inn=384) == BAD_SHAPE   # in % 256
    # grouped: null array, empty group, one bad member rejects the whole group
    assert lib.forge_wgrad_adamw_grouped(None, 1, *HP, 0, None) == NULL_PTR
    arr = (fb.forge_problem_t * 2)()
    for a in arr:
        a.X, a.dY, a.W, a.m, a.v, a.T, a.out, a.in_ = 0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 128, 384, 256
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
    assert lib.forge_wgrad_store_g(None, 0x2000, 0x3000, 128, 384, 256, None) == NULL_PTR
    assert lib.forge_adamw_from_g(None, 0x3000, 0x4000, 0x5000, None, None, 384, 256, *HP, 0, None) == NULL_PTR
    assert lib.forge_wgrad_adamw_host(0x1000, 0x2000, 0x3000, 0x4000, 0x5000, None, None, 0, 384, 256, *HP, 0) == BAD_SHAPE


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

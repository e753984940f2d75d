"""Thin ctypes binding of include/forge.h -- argument marshalling only; every step of the path
runs in the CUDA kernels of libforge_b200.so.  There is no fallback: if the library is missing
or a call fails, this module raises.

Tensors are torch CUDA tensors (PyTorch only allocates device memory and provides streams):
X [T,in] bf16, dY [T,out] bf16, W [out,in] bf16, m/v [out,in] in float32 | bfloat16 | int8+uint8,
scales [out,in/256] float32 for int8.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import c_float, c_int32, c_int64, c_void_p

import torch

from . import build as _build

FP32, BF16, INT8, FP8 = 0, 1, 2, 3
QBLOCK = 256
STATUS_NAMES = ["FORGE_OK", "FORGE_ERR_NULL_PTR", "FORGE_ERR_BAD_SHAPE", "FORGE_ERR_ALIGNMENT",
                "FORGE_ERR_BAD_HYPERPARAM", "FORGE_ERR_BAD_DTYPE", "FORGE_ERR_UNSUPPORTED_ARCH",
                "FORGE_ERR_CUDA", "FORGE_ERR_TOO_LARGE"]
NOALLOC_SCRATCH_BYTES = 32 << 20   # include/forge.h FORGE_NOALLOC_SCRATCH_BYTES
EXPORTS = ["forge_wgrad_adamw", "forge_wgrad_adamw_grouped", "forge_wgrad_step_grouped", "forge_wgrad_accumulate_grouped", "forge_layer_backward_grouped", "forge_wgrad_adamw_sr_grouped", "forge_wgrad_adamw_host", "forge_wgrad_adamw_host_noalloc", "forge_wgrad_adamw_grouped_host",
           "forge_wgrad_store_g", "forge_wgrad_store_g_grouped", "forge_adamw_from_g", "forge_workspace_bytes", "forge_launch_count",
           "forge_last_cuda_error", "forge_last_kernel", "forge_set_tuning", "forge_get_tuning", "forge_status_string", "forge_version"]


class ForgeError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        super().__init__(f"{where}: {name} (cuda error {lib().forge_last_cuda_error()})")


class forge_problem_t(ctypes.Structure):
    _fields_ = [("X", c_void_p), ("dY", c_void_p), ("W", c_void_p), ("m", c_void_p), ("v", c_void_p),
                ("m_scale", c_void_p), ("v_scale", c_void_p),
                ("T", c_int32), ("out", c_int32), ("in_", c_int32), ("ldx", c_int64), ("lddy", c_int64)]


class forge_opt_desc_t(ctypes.Structure):
    _fields_ = [("family", ctypes.c_int), ("nesterov", c_int32), ("step", c_int64),
                ("lr", c_float), ("beta1", c_float), ("beta2", c_float), ("eps", c_float), ("wd", c_float),
                ("momentum", c_float)]


FAMILIES = {"adamw": 0, "sgd": 1, "momentum": 2, "lion": 3, "rmsprop": 4, "adagrad": 5, "adamax": 6, "nadam": 7, "radam": 8}
FAMILY_STATES = {"adamw": 2, "sgd": 0, "momentum": 1, "lion": 1, "rmsprop": 1, "adagrad": 1, "adamax": 2, "nadam": 2, "radam": 2}

_lib = None
_libs = {}
_profiling = False


def use_profiling_library(on: bool) -> None:
    """Route every call of this module through libforge_b200_prof.so (the -DFORGE_PROFILING build: FORGE_CFG /
    FORGE_GRID / FORGE_ABLATE are honoured there and nowhere else).  For profiles/ commands and two tests only."""
    global _lib, _profiling
    if on and not os.path.exists(_build.PROF_LIB_PATH):
        _build.build(profiling=True)        # tests / profiles on a box that received only the product library
    _profiling = bool(on)
    _lib = None


def lib() -> ctypes.CDLL:
    """Load libforge_b200.so (built in-tree by build.build()); raises if it cannot be loaded."""
    global _lib
    if _lib is None and _profiling in _libs:
        _lib = _libs[_profiling]
    if _lib is None:
        path = _build.PROF_LIB_PATH if _profiling else _build.LIB_PATH
        if not os.path.exists(path):
            raise FileNotFoundError(f"{path} not built: run `python -m paper_2606_22932_b200.build"
                                    f"{' --profiling' if _profiling else ''}` (there is no fallback path)")
        L = ctypes.CDLL(path)
        hp = [c_int64, c_float, c_float, c_float, c_float, c_float]
        L.forge_wgrad_adamw.restype = ctypes.c_int
        L.forge_wgrad_adamw.argtypes = [c_void_p] * 7 + [c_int32] * 3 + hp + [ctypes.c_int, c_void_p]
        L.forge_wgrad_adamw_grouped.restype = ctypes.c_int
        L.forge_wgrad_adamw_grouped.argtypes = [ctypes.POINTER(forge_problem_t), c_int32] + hp + [ctypes.c_int, c_void_p]
        L.forge_wgrad_adamw_grouped_host.restype = ctypes.c_int
        L.forge_wgrad_adamw_grouped_host.argtypes = [ctypes.POINTER(forge_problem_t), c_int32] + hp + [ctypes.c_int]
        L.forge_wgrad_step_grouped.restype = ctypes.c_int
        L.forge_wgrad_step_grouped.argtypes = [ctypes.POINTER(forge_problem_t), c_int32, ctypes.POINTER(forge_opt_desc_t),
                                               ctypes.c_int, c_void_p]
        L.forge_wgrad_accumulate_grouped.restype = ctypes.c_int
        L.forge_wgrad_accumulate_grouped.argtypes = [ctypes.POINTER(forge_problem_t), c_int32, c_float, ctypes.c_int, c_void_p]
        L.forge_wgrad_adamw_sr_grouped.restype = ctypes.c_int
        L.forge_wgrad_adamw_sr_grouped.argtypes = [ctypes.POINTER(forge_problem_t), c_int32] + hp + \
                                                  [ctypes.c_int, ctypes.c_uint64, c_void_p]
        L.forge_layer_backward_grouped.restype = ctypes.c_int
        L.forge_layer_backward_grouped.argtypes = [ctypes.POINTER(forge_problem_t), ctypes.POINTER(c_void_p), c_int32] + hp + \
                                                  [ctypes.c_int, c_void_p]
        L.forge_wgrad_adamw_host.restype = ctypes.c_int
        L.forge_wgrad_adamw_host.argtypes = [c_void_p] * 7 + [c_int32] * 3 + hp + [ctypes.c_int]
        L.forge_wgrad_adamw_host_noalloc.restype = ctypes.c_int
        L.forge_wgrad_adamw_host_noalloc.argtypes = [c_void_p] * 7 + [c_int32] * 3 + hp + [ctypes.c_int]
        L.forge_wgrad_store_g.restype = ctypes.c_int
        L.forge_wgrad_store_g.argtypes = [c_void_p] * 3 + [c_int32] * 3 + [c_void_p]
        L.forge_wgrad_store_g_grouped.restype = ctypes.c_int
        L.forge_wgrad_store_g_grouped.argtypes = [ctypes.POINTER(forge_problem_t), c_int32, c_void_p]
        L.forge_adamw_from_g.restype = ctypes.c_int
        L.forge_adamw_from_g.argtypes = [c_void_p] * 6 + [c_int32] * 2 + hp + [ctypes.c_int, c_void_p]
        L.forge_workspace_bytes.restype = ctypes.c_size_t
        L.forge_launch_count.restype = ctypes.c_uint64
        L.forge_last_cuda_error.restype = ctypes.c_int
        L.forge_last_kernel.restype = ctypes.c_char_p
        L.forge_set_tuning.restype = ctypes.c_int
        L.forge_set_tuning.argtypes = [ctypes.c_int]
        L.forge_get_tuning.restype = ctypes.c_int
        L.forge_status_string.restype = ctypes.c_char_p
        L.forge_status_string.argtypes = [ctypes.c_int]
        L.forge_version.restype = ctypes.c_int
        _libs[_profiling] = L
        _lib = L
    return _lib


def _ptr(t):
    return None if t is None else c_void_p(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return c_void_p(s.cuda_stream)


def moment_dtype_of(m: torch.Tensor) -> int:
    return {torch.float32: FP32, torch.bfloat16: BF16, torch.int8: INT8, torch.uint8: FP8}[m.dtype]   # uint8 m = e4m3 codes


def _check(status: int, where: str):
    if status != 0:
        raise ForgeError(status, where)


def _dense(where: str, **tensors):
    """The single-problem entries and the state pointers of forge_problem_t carry no pitch: a strided view would be
    read as if it were dense.  Rejected here with the library's own BAD_SHAPE status."""
    for name, t in tensors.items():
        if t is not None and not t.is_contiguous():
            raise ForgeError(2, f"{where}: {name} must be contiguous (use the grouped entry for strided operand views)")


def forge_wgrad_adamw(X, dY, W, m, v, step, lr, beta1, beta2, eps, wd, m_scale=None, v_scale=None,
                      moment_dtype=None, stream=None, check=True) -> int:
    """include/forge.h forge_wgrad_adamw (Algorithm 1). In place on W, m, v."""
    _dense("forge_wgrad_adamw", X=X, dY=dY, W=W, m=m, v=v, m_scale=m_scale, v_scale=v_scale)
    T, inn = X.shape
    out = dY.shape[1]
    mdt = moment_dtype_of(m) if moment_dtype is None else moment_dtype
    st = lib().forge_wgrad_adamw(_ptr(X), _ptr(dY), _ptr(W), _ptr(m), _ptr(v), _ptr(m_scale), _ptr(v_scale),
                                 T, out, inn, int(step), lr, beta1, beta2, eps, wd, mdt, _stream(stream))
    if check:
        _check(st, "forge_wgrad_adamw")
    return st


def make_problem_array(problems):
    """problems: iterable of dicts/objects with X, dY, W, m, v (and m_scale, v_scale for int8)."""
    arr = (forge_problem_t * len(problems))()
    for i, p in enumerate(problems):
        g = p.get if isinstance(p, dict) else (lambda k, d=None, p=p: getattr(p, k, d))
        X, dY = g("X"), g("dY")
        arr[i].X, arr[i].dY = X.data_ptr(), dY.data_ptr()
        m, v, W = g("m"), g("v"), g("W")
        arr[i].W = None if W is None else W.data_ptr()
        arr[i].m = None if m is None else m.data_ptr()
        arr[i].v = None if v is None else v.data_ptr()
        ms, vs = g("m_scale"), g("v_scale")
        _dense("forge_problem_t", W=W, m=m, v=v, m_scale=ms, v_scale=vs)
        arr[i].m_scale = None if ms is None else ms.data_ptr()
        arr[i].v_scale = None if vs is None else vs.data_ptr()
        arr[i].T, arr[i].in_ = X.shape
        arr[i].out = dY.shape[1]
        # operands may be column slices of a wider tensor (fused QKV / gate-up): row pitch in elements, 0 = dense
        for t, name in ((X, "X"), (dY, "dY")):
            if t.dim() != 2 or (t.shape[1] > 1 and t.stride(1) != 1):
                raise ValueError(f"{name} must be a 2-D tensor with unit column stride")
        arr[i].ldx = 0 if X.is_contiguous() else X.stride(0)
        arr[i].lddy = 0 if dY.is_contiguous() else dY.stride(0)
    return arr


def forge_wgrad_adamw_grouped(problems, step, lr, beta1, beta2, eps, wd, moment_dtype, stream=None,
                              check=True, _arr=None) -> int:
    """include/forge.h forge_wgrad_adamw_grouped: all projections of a layer in one launch."""
    arr = make_problem_array(problems) if _arr is None else _arr
    st = lib().forge_wgrad_adamw_grouped(arr, len(arr), int(step), lr, beta1, beta2, eps, wd, moment_dtype,
                                         _stream(stream))
    if check:
        _check(st, "forge_wgrad_adamw_grouped")
    return st


def forge_wgrad_step_grouped(problems, family: str, step, lr, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.0, momentum=0.0,
                             nesterov=False, state_dtype=FP32, stream=None, check=True, _arr=None) -> int:
    """include/forge.h forge_wgrad_step_grouped: the other coordinate-wise families.
    Problems carry m / v only for the states the family has (None otherwise)."""
    arr = make_problem_array(problems) if _arr is None else _arr
    desc = forge_opt_desc_t(FAMILIES[family], int(bool(nesterov)), int(step), lr, beta1, beta2, eps, wd, momentum)
    st = lib().forge_wgrad_step_grouped(arr, len(arr), ctypes.byref(desc), state_dtype, _stream(stream))
    if check:
        _check(st, "forge_wgrad_step_grouped")
    return st


def forge_wgrad_adamw_sr_grouped(problems, step, lr, beta1, beta2, eps, wd, moment_dtype, seed, stream=None, check=True) -> int:
    """include/forge.h forge_wgrad_adamw_sr_grouped: AdamW with the stochastic-rounding store of W."""
    arr = make_problem_array(problems)
    st = lib().forge_wgrad_adamw_sr_grouped(arr, len(arr), int(step), lr, beta1, beta2, eps, wd, moment_dtype, int(seed),
                                            _stream(stream))
    if check:
        _check(st, "forge_wgrad_adamw_sr_grouped")
    return st


def forge_layer_backward_grouped(problems, dX, step, lr, beta1, beta2, eps, wd, moment_dtype, stream=None, check=True) -> int:
    """include/forge.h forge_layer_backward_grouped: dX[i] = dY_i W_i from the pre-update W, then the fused step."""
    arr = make_problem_array(problems)
    ptrs = (c_void_p * len(dX))(*[t.data_ptr() for t in dX])
    st = lib().forge_layer_backward_grouped(arr, ptrs, len(arr), int(step), lr, beta1, beta2, eps, wd, moment_dtype,
                                            _stream(stream))
    if check:
        _check(st, "forge_layer_backward_grouped")
    return st


def forge_wgrad_accumulate_grouped(problems, mu, state_dtype=FP32, stream=None, check=True) -> int:
    """include/forge.h forge_wgrad_accumulate_grouped: B <- mu*B + dY^T X in place; problems carry
    X, dY and m = B only."""
    arr = make_problem_array(problems)
    st = lib().forge_wgrad_accumulate_grouped(arr, len(arr), mu, state_dtype, _stream(stream))
    if check:
        _check(st, "forge_wgrad_accumulate_grouped")
    return st


def forge_wgrad_adamw_host(X, dY, W, m, v, step, lr, beta1, beta2, eps, wd, m_scale=None, v_scale=None,
                           check=True) -> int:
    """Host-buffer entry (CPU tensors, ideally pinned): H2D, fused step, D2H inside the call."""
    _dense("forge_wgrad_adamw_host", X=X, dY=dY, W=W, m=m, v=v, m_scale=m_scale, v_scale=v_scale)
    T, inn = X.shape
    out = dY.shape[1]
    st = lib().forge_wgrad_adamw_host(_ptr(X), _ptr(dY), _ptr(W), _ptr(m), _ptr(v), _ptr(m_scale), _ptr(v_scale),
                                      T, out, inn, int(step), lr, beta1, beta2, eps, wd, moment_dtype_of(m))
    if check:
        _check(st, "forge_wgrad_adamw_host")
    return st


def forge_wgrad_adamw_host_noalloc(X, dY, W, m, v, step, lr, beta1, beta2, eps, wd, m_scale=None, v_scale=None,
                                   check=True) -> int:
    """include/forge.h forge_wgrad_adamw_host_noalloc: the host-buffer entry that stages through the library's static
    32 MiB device array (no cudaMalloc / cudaFree); FORGE_ERR_TOO_LARGE beyond that."""
    _dense("forge_wgrad_adamw_host_noalloc", X=X, dY=dY, W=W, m=m, v=v, m_scale=m_scale, v_scale=v_scale)
    T, inn = X.shape
    out = dY.shape[1]
    st = lib().forge_wgrad_adamw_host_noalloc(_ptr(X), _ptr(dY), _ptr(W), _ptr(m), _ptr(v), _ptr(m_scale), _ptr(v_scale),
                                              T, out, inn, int(step), lr, beta1, beta2, eps, wd, moment_dtype_of(m))
    if check:
        _check(st, "forge_wgrad_adamw_host_noalloc")
    return st


def forge_wgrad_adamw_grouped_host(problems, step, lr, beta1, beta2, eps, wd, moment_dtype, check=True, _arr=None) -> int:
    """Host-buffer group entry (CPU tensors, ideally pinned): pipelined H2D / fused step / D2H per problem."""
    arr = make_problem_array(problems) if _arr is None else _arr
    st = lib().forge_wgrad_adamw_grouped_host(arr, len(arr), int(step), lr, beta1, beta2, eps, wd, moment_dtype)
    if check:
        _check(st, "forge_wgrad_adamw_grouped_host")
    return st


def forge_wgrad_store_g(X, dY, G, stream=None, check=True) -> int:
    """Store-G: G[out,in] fp32 = dY^T X; the DP bucket producer and the fused kernel's test twin."""
    _dense("forge_wgrad_store_g", X=X, dY=dY, G=G)
    T, inn = X.shape
    out = dY.shape[1]
    st = lib().forge_wgrad_store_g(_ptr(X), _ptr(dY), _ptr(G), T, out, inn, _stream(stream))
    if check:
        _check(st, "forge_wgrad_store_g")
    return st


def forge_wgrad_store_g_grouped(problems, stream=None, check=True, _arr=None) -> int:
    """include/forge.h forge_wgrad_store_g_grouped: problems carry X, dY and m = the fp32 G slice (dp.py buckets)."""
    arr = make_problem_array(problems) if _arr is None else _arr
    st = lib().forge_wgrad_store_g_grouped(arr, len(arr), _stream(stream))
    if check:
        _check(st, "forge_wgrad_store_g_grouped")
    return st


def forge_adamw_from_g(G, W, m, v, step, lr, beta1, beta2, eps, wd, m_scale=None, v_scale=None, stream=None,
                       check=True) -> int:
    """The update from a materialised fp32 G: dp.py's reduced bucket, and the fused kernel's test twin."""
    _dense("forge_adamw_from_g", G=G, W=W, m=m, v=v, m_scale=m_scale, v_scale=v_scale)
    out, inn = W.shape
    st = lib().forge_adamw_from_g(_ptr(G), _ptr(W), _ptr(m), _ptr(v), _ptr(m_scale), _ptr(v_scale), out, inn,
                                  int(step), lr, beta1, beta2, eps, wd, moment_dtype_of(m), _stream(stream))
    if check:
        _check(st, "forge_adamw_from_g")
    return st


TUNE_BOOST_CLOCK, TUNE_SUSTAINED_CLOCK = 0, 1


def forge_set_tuning(tuning: int) -> None:
    """include/forge.h forge_set_tuning: which clock the caller expects (bit-identical results either way)."""
    _check(lib().forge_set_tuning(int(tuning)), "forge_set_tuning")


def forge_get_tuning() -> int:
    return int(lib().forge_get_tuning())


def forge_launch_count() -> int:
    return int(lib().forge_launch_count())


def forge_workspace_bytes() -> int:
    return int(lib().forge_workspace_bytes())


def forge_version() -> int:
    return int(lib().forge_version())


def forge_status_string(status: int) -> str:
    return lib().forge_status_string(status).decode()

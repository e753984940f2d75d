"""TEST INFRASTRUCTURE ONLY -- numpy/ctypes front end of the CPU oracle in ``forge_oracle.c``.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It shares nothing with the CUDA path under
``paper_2606_22932_b200/`` and never imports it.  All arithmetic of the method lives in the C
file (each function there cites the PAPER.md passage it follows); this module only marshals
numpy arrays.  bf16 tensors are carried as ``uint16`` bit patterns.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import c_double, c_float, c_int, c_long, c_size_t, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "forge_oracle.c")
_SRC_FAM = os.path.join(_HERE, "forge_oracle_families.c")
_LIB = os.path.join(_HERE, "libforge_oracle.so")
QBLOCK = 256


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_FAM)):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", _LIB, _SRC, _SRC_FAM, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.forge_oracle_bf16_to_double.restype = c_double
        L.forge_oracle_bf16_to_double.argtypes = [ctypes.c_uint16]
        L.forge_oracle_bf16_from_double.restype = ctypes.c_uint16
        L.forge_oracle_bf16_from_double.argtypes = [c_double]
        L.forge_oracle_wgrad_rows.restype = None
        L.forge_oracle_wgrad_rows.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_long,
                                              c_long, c_int, c_int, c_void_p, c_void_p]
        hp = [c_long, c_float, c_float, c_float, c_float, c_float]
        dbg = [c_void_p, c_void_p, c_void_p]
        L.forge_oracle_adamw_fp32.restype = None
        L.forge_oracle_adamw_fp32.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_size_t] + hp + dbg
        L.forge_oracle_adamw_bf16.restype = None
        L.forge_oracle_adamw_bf16.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_size_t] + hp + dbg
        L.forge_oracle_adamw_int8.restype = None
        L.forge_oracle_adamw_int8.argtypes = [c_void_p] * 6 + [c_int, c_int] + hp + dbg
        L.forge_oracle_quant_matrix.restype = None
        L.forge_oracle_quant_matrix.argtypes = [c_void_p, c_void_p, c_int, c_int] + [c_void_p] * 4
        L.forge_oracle_bf16_from_double_array.restype = None
        L.forge_oracle_bf16_from_double_array.argtypes = [c_void_p, c_void_p, c_size_t]
        L.forge_oracle_num_threads.restype = c_int
        L.forge_oracle_sr_bits.restype = ctypes.c_uint32
        L.forge_oracle_sr_bits.argtypes = [ctypes.c_uint64, c_long, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32]
        L.forge_oracle_bf16_sr_from_double.restype = ctypes.c_uint16
        L.forge_oracle_bf16_sr_from_double.argtypes = [c_double, ctypes.c_uint32]
        L.forge_oracle_adamw_fp32_sr.restype = None
        L.forge_oracle_adamw_fp32_sr.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_int, c_long,
                                                 c_float, c_float, c_float, c_float, c_float, ctypes.c_uint64, ctypes.c_uint32]
        L.forge_oracle_e4m3_from_float.restype = ctypes.c_uint8
        L.forge_oracle_e4m3_from_float.argtypes = [c_float]
        L.forge_oracle_e4m3_to_double.restype = c_double
        L.forge_oracle_e4m3_to_double.argtypes = [ctypes.c_uint8]
        L.forge_oracle_fp8_quantize.restype = None
        L.forge_oracle_fp8_quantize.argtypes = [c_void_p, c_size_t, c_void_p, c_void_p]
        L.forge_oracle_adamw_fp8.restype = None
        L.forge_oracle_adamw_fp8.argtypes = [c_void_p] * 6 + [c_size_t, c_long, c_float, c_float, c_float, c_float, c_float]
        L.forge_oracle_accumulate.restype = None
        L.forge_oracle_accumulate.argtypes = [c_void_p, c_int, c_void_p, c_size_t, c_float]
        L.forge_oracle_family_step.restype = None
        L.forge_oracle_family_step.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_size_t,
                                               c_long, c_float, c_float, c_float, c_float, c_float, c_float,
                                               c_int, c_void_p]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(c_void_p)


def _chk(a, dtype, name):
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous):
        raise TypeError(f"{name}: expected C-contiguous numpy {np.dtype(dtype).name}")


def num_threads() -> int:
    return int(lib().forge_oracle_num_threads())


# ------------------------------------------------------------------ bf16 helpers -------------
def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    """uint16 bf16 bit patterns -> float64 (exact)."""
    _chk(bits, np.uint16, "bits")
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def f64_to_bf16(x: np.ndarray) -> np.ndarray:
    """float64 -> bf16 bits, one RNE rounding (forge_oracle_bf16_from_double)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty(x.shape, dtype=np.uint16)
    lib().forge_oracle_bf16_from_double_array(_p(x), _p(y), x.size)
    return y


# ------------------------------------------------------------------ gradient -----------------
def wgrad(dY: np.ndarray, X: np.ndarray, rows=None, with_abs: bool = False):
    """G = dY^T X in fp64, t ascending (Eq. 3).  dY [T,out], X [T,in] uint16 bf16 bits.

    ``rows=(p0,p1)`` restricts to output rows p0..p1-1 (exact for those rows).
    ``with_abs`` also returns E = |dY|^T |X| for the accumulation-error bound.
    """
    _chk(dY, np.uint16, "dY"); _chk(X, np.uint16, "X")
    T, out = dY.shape
    T2, inn = X.shape
    assert T == T2
    p0, p1 = (0, out) if rows is None else rows
    G = np.empty((p1 - p0, inn), dtype=np.float64)
    E = np.empty_like(G) if with_abs else None
    lib().forge_oracle_wgrad_rows(_p(dY), _p(X), T, out, inn, out, inn, p0, p1, _p(G), _p(E))
    return (G, E) if with_abs else G


# ------------------------------------------------------------------ AdamW --------------------
def adamw_fp32(W, m, v, G, step, lr, beta1, beta2, eps, wd, debug: bool = False):
    """In place: W uint16 bf16 bits, m/v float32 (Alg. 1 lines 6-11)."""
    _chk(W, np.uint16, "W"); _chk(m, np.float32, "m"); _chk(v, np.float32, "v"); _chk(G, np.float64, "G")
    assert W.shape == m.shape == v.shape == G.shape
    d = [np.empty(W.shape, np.float64) for _ in range(3)] if debug else [None] * 3
    lib().forge_oracle_adamw_fp32(_p(W), _p(m), _p(v), _p(G), W.size, int(step), lr, beta1, beta2,
                                  eps, wd, _p(d[0]), _p(d[1]), _p(d[2]))
    return tuple(d) if debug else None


def adamw_bf16(W, m, v, G, step, lr, beta1, beta2, eps, wd, debug: bool = False):
    """In place: W, m, v all uint16 bf16 bits."""
    for a, n in ((W, "W"), (m, "m"), (v, "v")):
        _chk(a, np.uint16, n)
    _chk(G, np.float64, "G")
    assert W.shape == m.shape == v.shape == G.shape
    d = [np.empty(W.shape, np.float64) for _ in range(3)] if debug else [None] * 3
    lib().forge_oracle_adamw_bf16(_p(W), _p(m), _p(v), _p(G), W.size, int(step), lr, beta1, beta2,
                                  eps, wd, _p(d[0]), _p(d[1]), _p(d[2]))
    return tuple(d) if debug else None


def adamw_int8(W, mq, vq, m_scale, v_scale, G, step, lr, beta1, beta2, eps, wd, debug: bool = False):
    """In place: W uint16; mq int8, vq uint8 [out,in]; scales float32 [out,in/256]."""
    _chk(W, np.uint16, "W"); _chk(mq, np.int8, "mq"); _chk(vq, np.uint8, "vq")
    _chk(m_scale, np.float32, "m_scale"); _chk(v_scale, np.float32, "v_scale"); _chk(G, np.float64, "G")
    out, inn = W.shape
    assert inn % QBLOCK == 0 and m_scale.shape == v_scale.shape == (out, inn // QBLOCK)
    d = [np.empty(W.shape, np.float64) for _ in range(3)] if debug else [None] * 3
    lib().forge_oracle_adamw_int8(_p(W), _p(mq), _p(vq), _p(m_scale), _p(v_scale), _p(G), out, inn,
                                  int(step), lr, beta1, beta2, eps, wd, _p(d[0]), _p(d[1]), _p(d[2]))
    return tuple(d) if debug else None


def quantize(m: np.ndarray | None, v: np.ndarray | None):
    """Blockwise int8 quantiser (256 along `in`): returns (mq, m_scale, vq, v_scale)."""
    ref = m if m is not None else v
    out, inn = ref.shape
    assert inn % QBLOCK == 0
    md = None if m is None else np.ascontiguousarray(m, dtype=np.float64)
    vd = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
    mq = np.zeros((out, inn), np.int8); vq = np.zeros((out, inn), np.uint8)
    ms = np.zeros((out, inn // QBLOCK), np.float32); vs = np.zeros((out, inn // QBLOCK), np.float32)
    lib().forge_oracle_quant_matrix(_p(md), _p(vd), out, inn, _p(mq), _p(vq), _p(ms), _p(vs))
    return mq, ms, vq, vs


def dequantize_m(mq: np.ndarray, m_scale: np.ndarray) -> np.ndarray:
    return mq.astype(np.float64) * np.repeat(m_scale.astype(np.float64) / 127.0, QBLOCK, axis=1)


def dequantize_v(vq: np.ndarray, v_scale: np.ndarray) -> np.ndarray:
    return vq.astype(np.float64) * np.repeat(v_scale.astype(np.float64) / 255.0, QBLOCK, axis=1)


def step_fp32(dY, X, W, m, v, step, lr, beta1, beta2, eps, wd):
    """One whole hot-path step with fp32 moments: G then AdamW, in place."""
    adamw_fp32(W, m, v, wgrad(dY, X), step, lr, beta1, beta2, eps, wd)


# ------------------------------------------------------------------ other regime-1 families --
FAMILIES = {"sgd": 1, "momentum": 2, "lion": 3, "rmsprop": 4, "adagrad": 5, "adamax": 6, "nadam": 7, "radam": 8}
FAMILY_STATES = {"sgd": 0, "momentum": 1, "lion": 1, "rmsprop": 1, "adagrad": 1, "adamax": 2, "nadam": 2, "radam": 2}


def family_step(family: str, W, s0, s1, G, step, lr, beta1=0.9, beta2=0.999, eps=1e-8, wd=0.0, momentum=0.0,
                nesterov=False, debug: bool = False):
    """In place step of one coordinate-wise family (forge_oracle_families.c).
    W uint16 bf16 bits; s0/s1 float32 or uint16 (bf16 bits) arrays or None; G float64."""
    _chk(W, np.uint16, "W"); _chk(G, np.float64, "G")
    ns = FAMILY_STATES[family]
    states = [s0, s1][:ns]
    assert all(s is not None for s in states) and all(s is None for s in [s0, s1][ns:])
    bf16 = bool(states) and states[0].dtype == np.uint16
    for s in states:
        _chk(s, np.uint16 if bf16 else np.float32, "state")
        assert s.shape == W.shape
    Wd = np.empty(W.shape, np.float64) if debug else None
    lib().forge_oracle_family_step(FAMILIES[family], _p(W), _p(s0), _p(s1), int(bf16), _p(G), W.size, int(step),
                                   lr, beta1, beta2, eps, wd, momentum, int(bool(nesterov)), _p(Wd))
    return Wd


def accumulate(B, G, mu):
    """In place B <- mu*B + G (Muon's A-step); B float32 or uint16 bf16 bits, G float64."""
    _chk(G, np.float64, "G")
    bf16 = B.dtype == np.uint16
    _chk(B, np.uint16 if bf16 else np.float32, "B")
    assert B.shape == G.shape
    lib().forge_oracle_accumulate(_p(B), int(bf16), _p(G), B.size, mu)


# ------------------------------------------------------------------ input gradient ----------
def dgrad(dY: np.ndarray, W: np.ndarray) -> np.ndarray:
    """dX = dY . W from the PRE-update W (Algorithm 1 line 1), the plain definition:
    dX[t,q] = sum_p dY[t,p] W[p,q] in fp64 (numpy matmul as the library primitive).  dY [T,out], W [out,in]
    uint16 bf16 bits; returns float64 [T,in] (round with f64_to_bf16 for the stored bf16 dX)."""
    _chk(dY, np.uint16, "dY"); _chk(W, np.uint16, "W")
    return bf16_to_f64(dY) @ bf16_to_f64(W)


# ------------------------------------------------------------------ stochastic-rounding store
def sr_bits(seed, step, stream, row, col) -> int:
    """The 16 random bits of weight element (row, col) (forge_oracle_families.c, reading S16)."""
    return int(lib().forge_oracle_sr_bits(int(seed), int(step), int(stream), int(row), int(col)))


def bf16_sr(x: float, r16: int) -> int:
    return int(lib().forge_oracle_bf16_sr_from_double(float(x), int(r16)))


def adamw_fp32_sr(W, m, v, G, step, lr, beta1, beta2, eps, wd, seed, stream=0):
    """AdamW with fp32 moments and the stochastic-rounding store of W, in place."""
    _chk(W, np.uint16, "W"); _chk(m, np.float32, "m"); _chk(v, np.float32, "v"); _chk(G, np.float64, "G")
    assert W.ndim == 2 and W.shape == m.shape == v.shape == G.shape
    lib().forge_oracle_adamw_fp32_sr(_p(W), _p(m), _p(v), _p(G), W.shape[0], W.shape[1], int(step), lr, beta1, beta2,
                                     eps, wd, int(seed), int(stream))


# ------------------------------------------------------------------ fp8 (e4m3) moments ------
def e4m3_from_float(t: float) -> int:
    return int(lib().forge_oracle_e4m3_from_float(float(np.float32(t))))


def e4m3_to_double(code: int) -> float:
    return float(lib().forge_oracle_e4m3_to_double(int(code)))


def fp8_quantize(x: np.ndarray):
    """fp32 tensor -> (e4m3 codes uint8, scale float32[2] = [amax/448, 0]) (reading S17)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    code = np.empty(x.shape, np.uint8)
    scale = np.zeros(2, np.float32)
    lib().forge_oracle_fp8_quantize(_p(x), x.size, _p(code), _p(scale))
    return code, scale


def fp8_dequantize(code: np.ndarray, scale) -> np.ndarray:
    lut = np.array([e4m3_to_double(c) for c in range(256)])
    return lut[code] * float(scale[0])


def adamw_fp8(W, mq, vq, m_scale, v_scale, G, step, lr, beta1, beta2, eps, wd):
    """In place AdamW with e4m3 moments, per-tensor delayed scaling (reading S17).
    m_scale / v_scale float32[2]: [0] scale in use, [1] amax of this step's m' / v' (max-accumulated)."""
    _chk(W, np.uint16, "W"); _chk(mq, np.uint8, "mq"); _chk(vq, np.uint8, "vq"); _chk(G, np.float64, "G")
    _chk(m_scale, np.float32, "m_scale"); _chk(v_scale, np.float32, "v_scale")
    assert W.shape == mq.shape == vq.shape == G.shape and m_scale.shape == v_scale.shape == (2,)
    lib().forge_oracle_adamw_fp8(_p(W), _p(mq), _p(vq), _p(m_scale), _p(v_scale), _p(G), W.size, int(step),
                                 lr, beta1, beta2, eps, wd)

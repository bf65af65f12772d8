"""CPU oracle for the chained GEMM Y = act(X.W1).W2.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_2607_07862_b200) never imports this, and this never imports the binding.

Two independent implementations live here:
  * `oracle_mlp.c`  -- the oracle proper (C, OpenMP), loaded through ctypes;
  * `brute_*`       -- pure-Python exact-rational / integer brute force for tiny
                       shapes, used only to pin the C oracle (tests/test_oracle_pins.py).
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from fractions import Fraction
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_mlp.c")

ACT_NONE, ACT_RELU, ACT_GELU_TANH = 0, 1, 2


def _cpu_tag() -> str:
    """The .so is compiled -march=native; key it by the host's ISA flags so a
    library built on one machine is never loaded on a different CPU."""
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


def lib_path() -> str:
    return os.path.join(_HERE, f"liboracle_{_cpu_tag()}.so")


def build(force: bool = False) -> str:
    """Compile oracle_mlp.c with gcc (no -ffast-math, no fp contraction)."""
    out = lib_path()
    if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
        return out
    cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fno-fast-math", "-ffp-contract=off",
           "-shared", "-fPIC", "-o", out, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return out


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u16p = ctypes.POINTER(ctypes.c_uint16)
        lib.oracle_bf16_to_f32.restype = ctypes.c_float
        lib.oracle_bf16_to_f32.argtypes = [ctypes.c_uint16]
        lib.oracle_bf16_rne.restype = ctypes.c_uint16
        lib.oracle_bf16_rne.argtypes = [ctypes.c_float]
        lib.oracle_gelu_tanh.restype = ctypes.c_float
        lib.oracle_gelu_tanh.argtypes = [ctypes.c_float]
        lib.oracle_act.restype = ctypes.c_float
        lib.oracle_act.argtypes = [ctypes.c_float, ctypes.c_int]
        lib.oracle_gemm_layer.restype = ctypes.c_int
        lib.oracle_gemm_layer.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, u16p, u16p, ctypes.c_int,
                                          u16p, ctypes.POINTER(ctypes.c_float),
                                          ctypes.POINTER(ctypes.c_int64), ctypes.c_int]
        lib.oracle_mlp_chain.restype = ctypes.c_int
        lib.oracle_mlp_chain.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int), u16p,
                                         ctypes.POINTER(u16p), ctypes.c_int, ctypes.POINTER(u16p),
                                         ctypes.POINTER(ctypes.c_int64), ctypes.c_int]
        lib.oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _u16p(a: np.ndarray):
    assert a.dtype == np.uint16 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint16))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def bf16_rne(x: float) -> int:
    return int(_load().oracle_bf16_rne(ctypes.c_float(x)))


def bf16_to_f32(h: int) -> float:
    return float(_load().oracle_bf16_to_f32(ctypes.c_uint16(h)))


def gelu_tanh(x: float) -> float:
    return float(_load().oracle_gelu_tanh(ctypes.c_float(x)))


def act_f32(x: float, act: int) -> float:
    return float(_load().oracle_act(ctypes.c_float(x), act))


def gemm_layer(A: np.ndarray, W: np.ndarray, act: int, want_acc: bool = False, want_cert: bool = False,
               threads: int = 0):
    """One layer: A [M x K] u16(bf16), W [N x K] u16(bf16) -> out [M x N] u16(bf16).

    Returns (out, acc or None, cert or None); cert = (max |partial| in int64,
    #accumulators where fp32 != int64, non-integer-operand flag)."""
    A = np.ascontiguousarray(A, dtype=np.uint16)
    W = np.ascontiguousarray(W, dtype=np.uint16)
    M, K = A.shape
    N, K2 = W.shape
    assert K == K2, "W must be [N x K], K contiguous"
    out = np.empty((M, N), dtype=np.uint16)
    acc = np.empty((M, N), dtype=np.float32) if want_acc else None
    cert = (ctypes.c_int64 * 3)() if want_cert else None
    rc = _load().oracle_gemm_layer(M, K, N, _u16p(A), _u16p(W), act, _u16p(out),
                                   acc.ctypes.data_as(ctypes.POINTER(ctypes.c_float)) if want_acc else None,
                                   cert, threads)
    if rc:
        raise RuntimeError(f"oracle_gemm_layer failed: {rc}")
    return out, acc, (tuple(int(c) for c in cert) if want_cert else None)


def mlp_chain(X: np.ndarray, Ws: Sequence[np.ndarray], act: int, want_cert: bool = False, threads: int = 0):
    """The whole chain.  X [M x K] u16, Ws[l] [N_l x K_l] u16.

    Returns (outs, certs): outs[l] is A^{l+1} ([M x N_{l+1}] u16); outs[-1] is Y.
    certs is a list of per-layer (max|partial|, #mismatch, nonint) or None."""
    X = np.ascontiguousarray(X, dtype=np.uint16)
    Ws = [np.ascontiguousarray(w, dtype=np.uint16) for w in Ws]
    M, K = X.shape
    L = len(Ws)
    widths = [K] + [w.shape[0] for w in Ws]
    for l, w in enumerate(Ws):
        assert w.shape[1] == widths[l], f"W[{l}] must be [N x K] with K={widths[l]}"
    outs = [np.empty((M, widths[l + 1]), dtype=np.uint16) for l in range(L)]
    u16p = ctypes.POINTER(ctypes.c_uint16)
    Wp = (u16p * L)(*[_u16p(w) for w in Ws])
    Op = (u16p * L)(*[_u16p(o) for o in outs])
    wd = (ctypes.c_int * (L + 1))(*widths)
    cert = (ctypes.c_int64 * (3 * L))() if want_cert else None
    rc = _load().oracle_mlp_chain(M, L, wd, _u16p(X), Wp, act, Op, cert, threads)
    if rc:
        raise RuntimeError(f"oracle_mlp_chain failed: {rc}")
    certs = [tuple(int(cert[3 * l + i]) for i in range(3)) for l in range(L)] if want_cert else None
    return outs, certs


# --------------------------------------------------------------------------
# Error metric of the parity bar (reading c3; BASELINE.json north_star
# "max relative error 2e-2"): err = max_ij |Yg - Yo| / max(|Yo_ij|, rms(Yo)).
# --------------------------------------------------------------------------
def u16_to_f64(a: np.ndarray) -> np.ndarray:
    return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def rel_err(got_u16: np.ndarray, ref_u16: np.ndarray) -> dict:
    g, r = u16_to_f64(np.ascontiguousarray(got_u16)), u16_to_f64(np.ascontiguousarray(ref_u16))
    if g.size == 0:
        return {"err": 0.0, "normwise": 0.0, "fro": 0.0, "nan": 0}
    nan = int(np.isnan(g).sum())
    d = np.abs(g - r)
    rms = float(np.sqrt(np.mean(r * r)))
    denom = np.maximum(np.abs(r), rms if rms > 0 else 1.0)
    return {
        "err": float(np.nanmax(d / denom)) if nan < g.size else float("inf"),
        "normwise": float(np.nanmax(d) / max(float(np.abs(r).max()), 1e-300)),
        "fro": float(np.sqrt(np.nansum(d * d)) / max(float(np.sqrt((r * r).sum())), 1e-300)),
        "nan": nan,
    }


# --------------------------------------------------------------------------
# Pure-Python brute force (tiny shapes only).  Independent of the C code: it
# works on exact rationals and only rounds where the definition rounds.
# --------------------------------------------------------------------------
def brute_bf16_value(h: int) -> Fraction:
    """Exact value of a (finite) bf16 bit pattern."""
    s = -1 if (h >> 15) & 1 else 1
    e = (h >> 7) & 0xFF
    f = h & 0x7F
    assert e != 0xFF, "finite only"
    if e == 0:
        return s * Fraction(f, 1 << 7) * Fraction(2) ** (-126)
    return s * (1 + Fraction(f, 1 << 7)) * Fraction(2) ** (e - 127)


def _round_to_precision(x: Fraction, p: int, emin: int) -> Fraction:
    """Round an exact rational to a binary float with p significand bits and minimum
    normal exponent emin, ties to even (no overflow handling: tiny inputs only)."""
    if x == 0:
        return Fraction(0)
    s = -1 if x < 0 else 1
    ax = abs(x)
    e = ax.numerator.bit_length() - ax.denominator.bit_length()
    if Fraction(2) ** e > ax:
        e -= 1
    if Fraction(2) ** (e + 1) <= ax:
        e += 1
    e = max(e, emin)
    ulp = Fraction(2) ** (e - (p - 1))
    q = ax / ulp
    fl = q.numerator // q.denominator
    rem = q - fl
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (fl & 1)):
        fl += 1
    return s * fl * ulp


def brute_round_f32(x: Fraction) -> Fraction:
    return _round_to_precision(x, 24, -126)


def brute_round_bf16(x: Fraction) -> Fraction:
    return _round_to_precision(x, 8, -126)


def brute_bf16_bits(x: Fraction) -> int:
    """bf16 bit pattern of an exactly representable value."""
    if x == 0:
        return 0
    s = 0x8000 if x < 0 else 0
    ax = abs(x)
    e = 0
    while Fraction(2) ** (e + 1) <= ax:
        e += 1
    while Fraction(2) ** e > ax:
        e -= 1
    if e < -126:
        f = ax / Fraction(2) ** (-126 - 7)
        assert f.denominator == 1
        return s | int(f)
    f = (ax / Fraction(2) ** e - 1) * 128
    assert f.denominator == 1, "not a bf16 value"
    return s | ((e + 127) << 7) | int(f)


def brute_mlp(X: List[List[int]], Ws: List[List[List[int]]], act: int) -> List[List[List[int]]]:
    """Chain on bf16 bit patterns with exact rationals, rounding only where the
    definition rounds: each fp32 add (RN-even), then act, then bf16 (RN-even).
    act must be NONE or RELU here (GeLU has its own pins).  W[l] is [N x K]."""
    assert act in (ACT_NONE, ACT_RELU)
    A = [[brute_bf16_value(h) for h in row] for row in X]
    outs = []
    L = len(Ws)
    for l, W in enumerate(Ws):
        Wv = [[brute_bf16_value(h) for h in row] for row in W]
        nxt, bits = [], []
        for m in range(len(A)):
            row_v, row_b = [], []
            for n in range(len(Wv)):
                acc = Fraction(0)
                for k in range(len(A[m])):
                    acc = brute_round_f32(acc + A[m][k] * Wv[n][k])
                if l < L - 1 and act == ACT_RELU and acc < 0:
                    acc = Fraction(0)
                v = brute_round_bf16(acc)
                row_v.append(v)
                row_b.append(brute_bf16_bits(v))
            nxt.append(row_v)
            bits.append(row_b)
        outs.append(bits)
        A = nxt
    return outs

"""ctypes binding of include/mlp_pipe.h -- argument marshalling only.

Every step of the path (ticketing, both GEMMs, activation, rounding, publish / poll) runs in the
CUDA kernels behind the C ABI; this module only turns torch tensors and streams into pointers.
There is NO CPU fallback: if csrc/libmlp_pipe.so is missing or the device is not sm_100 the
calls raise.  This module never imports `oracle/`.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

from . import build as _build

MLP_OK, MLP_ERR_INVALID, MLP_ERR_UNSUPPORTED, MLP_ERR_CUDA, MLP_ERR_OOM, MLP_ERR_TIMEOUT = range(6)
MLP_BF16 = 0
MLP_ACT_NONE, MLP_ACT_RELU, MLP_ACT_GELU_TANH = 0, 1, 2
MLP_SEQUENTIAL, MLP_MICROBATCH, MLP_CTA_PIPELINED = 0, 1, 2
MLP_MAX_LAYERS = 8
MLP_FLAG_TILE_MAJOR, MLP_FLAG_DEBUG_DELAY, MLP_FLAG_DEBUG_REVERSE, MLP_FLAG_NO_W_EVICT_FIRST = 1, 2, 4, 8
MLP_FLAG_AUTOTUNE = 0x400
MLP_FLAG_PDL = 0x800
MLP_FLAG_WORKQUEUE = 0x1000
MLP_FLAG_PAIR = 0x2000
MLP_FLAG_DEBUG_DROP_PUBLISH = 0x4000
MLP_FLAG_NO_COOPERATIVE = 0x8000
MLP_FLAG_MB_CORESIDENT = 0x10000
MLP_FLAG_TWO_KERNEL = 0x20000
MLP_FLAG_ACQUIRE_LOADS, MLP_FLAG_EXP_NO_ACQUIRE_FENCE, MLP_FLAG_EXP_NO_PROXY_FENCE = 0x40, 0x10, 0x20
MLP_FLAG_EXP_NO_FAST_PATH, MLP_FLAG_EXP_NO_PREISSUE = 0x80, 0x100

EXPORTS = [
    "mlp_pipe_create", "mlp_pipe_create_chain", "mlp_pipe_run", "mlp_pipe_run_chain", "mlp_pipe_run_host",
    "mlp_pipe_hidden", "mlp_pipe_poison_hidden", "mlp_pipe_stats", "mlp_pipe_destroy", "mlp_status_string",
    "mlp_pipe_last_error", "mlp_pipe_version", "mlp_pipe_cta_records", "mlp_pipe_plan", "mlp_pipe_plan_units",
    "mlp_pipe_run_static",
]
MLP_STATIC_SCRATCH_BYTES = 32 << 20


class mlp_mode(ctypes.Structure):
    _fields_ = [
        ("kind", ctypes.c_int), ("chunks", ctypes.c_int), ("sm_split", ctypes.c_float),
        ("tile_m", ctypes.c_int), ("tile_n", ctypes.c_int), ("tile_k", ctypes.c_int),
        ("stages", ctypes.c_int), ("kslice_tiles", ctypes.c_int), ("split_k", ctypes.c_int),
        ("flags", ctypes.c_uint), ("split_k_layer", ctypes.c_int * MLP_MAX_LAYERS),
        ("grid", ctypes.c_int), ("w_group", ctypes.c_int), ("timeout_ms", ctypes.c_int), ("a_stages", ctypes.c_int),
    ]


class mlp_stats(ctypes.Structure):
    _fields_ = [
        ("n_layers", ctypes.c_int), ("grid", ctypes.c_int), ("stages", ctypes.c_int), ("tile_m", ctypes.c_int),
        ("split_k", ctypes.c_int * MLP_MAX_LAYERS), ("units", ctypes.c_int * MLP_MAX_LAYERS),
        ("producer_ctas", ctypes.c_int), ("status", ctypes.c_uint32), ("runs", ctypes.c_uint64),
        ("flag_stall_cycles_sum", ctypes.c_uint64), ("flag_stall_cycles_max", ctypes.c_uint64),
        ("flag_polls", ctypes.c_uint64), ("kernel_cycles_max", ctypes.c_uint64),
        ("units_done", ctypes.c_uint32 * MLP_MAX_LAYERS),
        ("units_by_consumer_ctas", ctypes.c_uint32 * MLP_MAX_LAYERS), ("ready_ok", ctypes.c_uint32),
        ("tile_n", ctypes.c_int), ("reduce_mode", ctypes.c_int * MLP_MAX_LAYERS),
    ]


class mlp_cta_record(ctypes.Structure):
    _fields_ = [
        ("flag_stall_cycles", ctypes.c_uint64), ("flag_polls", ctypes.c_uint64), ("cycles", ctypes.c_uint64),
        ("ts", ctypes.c_uint64 * 8), ("wait", ctypes.c_uint64 * 8), ("units", ctypes.c_uint32 * MLP_MAX_LAYERS),
        ("unit_ts", (ctypes.c_uint64 * 4) * 12), ("unit_id", ctypes.c_uint32 * 12),
    ]


class mlp_plan(ctypes.Structure):
    _fields_ = [
        ("tile_m", ctypes.c_int), ("tile_n", ctypes.c_int), ("m_blks", ctypes.c_int), ("stages", ctypes.c_int),
        ("a_stages", ctypes.c_int), ("acc_stages", ctypes.c_int), ("grid", ctypes.c_int), ("producer_ctas", ctypes.c_int),
        ("smem_bytes", ctypes.c_int),
        ("tiles", ctypes.c_int * MLP_MAX_LAYERS), ("split_k", ctypes.c_int * MLP_MAX_LAYERS),
        ("reduce_mode", ctypes.c_int * MLP_MAX_LAYERS), ("ready_inc", ctypes.c_int * MLP_MAX_LAYERS),
        ("units", ctypes.c_int * MLP_MAX_LAYERS), ("model_us", ctypes.c_double),
    ]


class mlp_unit(ctypes.Structure):
    _fields_ = [("tile", ctypes.c_uint16), ("kind", ctypes.c_uint8), ("k_slice", ctypes.c_uint8),
                ("begin", ctypes.c_uint16), ("end", ctypes.c_uint16)]


_lib = None


def lib_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True):
    """dlopen csrc/libmlp_pipe.so (building it first if it is missing and nvcc is here)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        if not build_if_missing:
            raise RuntimeError(f"{path} is missing: run `python -m paper_2607_07862_b200.build`")
        _build.build_lib()
    lib = ctypes.CDLL(path)
    vp, ci = ctypes.c_void_p, ctypes.c_int
    lib.mlp_pipe_create.restype = ci
    lib.mlp_pipe_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, ci, ctypes.POINTER(mlp_mode)]
    lib.mlp_pipe_create_chain.restype = ci
    lib.mlp_pipe_create_chain.argtypes = [ctypes.POINTER(vp), ci, ci, ctypes.POINTER(ci), ci, ci, ctypes.POINTER(mlp_mode)]
    lib.mlp_pipe_run.restype = ci
    lib.mlp_pipe_run.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.mlp_pipe_run_chain.restype = ci
    lib.mlp_pipe_run_chain.argtypes = [vp, vp, ctypes.POINTER(vp), vp, vp]
    lib.mlp_pipe_run_host.restype = ci
    lib.mlp_pipe_run_host.argtypes = [vp, vp, ctypes.POINTER(vp), vp, vp, ctypes.POINTER(ctypes.c_size_t),
                                      ctypes.POINTER(ctypes.c_size_t)]
    lib.mlp_pipe_hidden.restype = ci
    lib.mlp_pipe_hidden.argtypes = [vp, ci, ctypes.POINTER(vp), ctypes.POINTER(ctypes.c_size_t)]
    lib.mlp_pipe_poison_hidden.restype = ci
    lib.mlp_pipe_poison_hidden.argtypes = [vp, ctypes.c_uint16, vp]
    lib.mlp_pipe_stats.restype = ci
    lib.mlp_pipe_stats.argtypes = [vp, ctypes.POINTER(mlp_stats), ctypes.c_size_t]
    lib.mlp_pipe_cta_records.restype = ci
    lib.mlp_pipe_cta_records.argtypes = [vp, ci, ctypes.POINTER(mlp_cta_record), ci, ctypes.POINTER(ci)]
    lib.mlp_pipe_plan.restype = ci
    lib.mlp_pipe_plan.argtypes = [ci, ci, ctypes.POINTER(ci), ctypes.POINTER(mlp_mode), ci, ctypes.POINTER(mlp_plan)]
    lib.mlp_pipe_plan_units.restype = ci
    lib.mlp_pipe_plan_units.argtypes = [ci, ci, ctypes.POINTER(ci), ctypes.POINTER(mlp_mode), ci, ci, ctypes.POINTER(mlp_unit), ci,
                                        ctypes.POINTER(ci)]
    lib.mlp_pipe_run_static.restype = ci
    lib.mlp_pipe_run_static.argtypes = [ci, ci, ctypes.POINTER(ci), ci, vp, ctypes.POINTER(vp), vp, vp]
    lib.mlp_pipe_destroy.restype = None
    lib.mlp_pipe_destroy.argtypes = [vp]
    lib.mlp_status_string.restype = ctypes.c_char_p
    lib.mlp_status_string.argtypes = [ci]
    lib.mlp_pipe_last_error.restype = ctypes.c_char_p
    lib.mlp_pipe_last_error.argtypes = [vp]
    lib.mlp_pipe_version.restype = ctypes.c_char_p
    lib.mlp_pipe_version.argtypes = []
    _lib = lib
    return lib


class MlpError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"mlp_pipe status {status} ({msg})")
        self.status = status


def _check(status: int, handle=None):
    if status != MLP_OK:
        lib = load()
        detail = lib.mlp_pipe_last_error(handle).decode() or lib.mlp_status_string(status).decode()
        raise MlpError(status, detail)


def make_mode(kind: int = MLP_CTA_PIPELINED, chunks: int = 0, sm_split: float = 1.0, tile_m: int = 0, stages: int = 0,
              split_k: int = 0, split_k_layer: Sequence[int] = (), flags: int = 0, grid: int = 0,
              timeout_ms: int = 0, w_group: int = 0, tile_n: int = 0, a_stages: int = 0) -> mlp_mode:
    m = mlp_mode()
    m.kind, m.chunks, m.sm_split, m.tile_m, m.stages = kind, chunks, sm_split, tile_m, stages
    m.tile_n = tile_n
    m.a_stages = a_stages
    m.split_k, m.flags, m.grid, m.timeout_ms = split_k, flags, grid, timeout_ms
    m.w_group = w_group
    for i, s in enumerate(split_k_layer):
        m.split_k_layer[i] = int(s)
    return m


def _stream_ptr(stream: Optional[torch.cuda.Stream]):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _dev_ptr(t: torch.Tensor, shape, name: str):
    if not t.is_cuda or t.dtype != torch.bfloat16 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: need a contiguous CUDA bf16 tensor of shape {tuple(shape)}, got {t.dtype} {tuple(t.shape)} {t.device}")
    return ctypes.c_void_p(t.data_ptr())


class MlpPipe:
    """Owner of one `mlp_pipe*`.  Thin: create / run / stats / hidden / destroy."""

    def __init__(self, M: int, widths: Sequence[int], act: int, mode: Optional[mlp_mode] = None):
        if not torch.cuda.is_available():
            raise RuntimeError("mlp_pipe needs a CUDA device (sm_100a); there is no CPU fallback")
        self._lib = load()
        self.M, self.widths, self.act = int(M), [int(w) for w in widths], int(act)
        self.L = len(self.widths) - 1
        self._h = ctypes.c_void_p()
        mp = ctypes.byref(mode) if mode is not None else None
        if self.L == 2:
            st = self._lib.mlp_pipe_create(ctypes.byref(self._h), self.M, self.widths[0], self.widths[1], self.widths[2],
                                           MLP_BF16, self.act, mp)
        else:
            w = (ctypes.c_int * (self.L + 1))(*self.widths)
            st = self._lib.mlp_pipe_create_chain(ctypes.byref(self._h), self.M, self.L, w, MLP_BF16, self.act, mp)
        if st != MLP_OK:
            self._h = ctypes.c_void_p()
            _check(st, None)

    def run(self, X: torch.Tensor, Ws: Sequence[torch.Tensor], Y: Optional[torch.Tensor] = None,
            stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        if len(Ws) != self.L:
            raise ValueError(f"need {self.L} weight tensors")
        if Y is None:
            Y = torch.empty((self.M, self.widths[-1]), dtype=torch.bfloat16, device=X.device)
        xp = _dev_ptr(X, (self.M, self.widths[0]), "X")
        yp = _dev_ptr(Y, (self.M, self.widths[-1]), "Y")
        wp = [_dev_ptr(w, (self.widths[l + 1], self.widths[l]), f"W[{l}]") for l, w in enumerate(Ws)]
        if self.L == 2:
            st = self._lib.mlp_pipe_run(self._h, xp, wp[0], wp[1], yp, _stream_ptr(stream))
        else:
            arr = (ctypes.c_void_p * self.L)(*wp)
            st = self._lib.mlp_pipe_run_chain(self._h, xp, arr, yp, _stream_ptr(stream))
        _check(st, self._h)
        return Y

    def run_host(self, X: torch.Tensor, Ws: Sequence[torch.Tensor], Y: torch.Tensor,
                 stream: Optional[torch.cuda.Stream] = None):
        """Host-buffer entry point (bench.py's e2e leg).  Returns (h2d_bytes, d2h_bytes)."""
        for t in [X, Y] + list(Ws):
            if t.is_cuda or t.dtype != torch.bfloat16 or not t.is_contiguous():
                raise ValueError("run_host needs contiguous CPU bf16 tensors")
        arr = (ctypes.c_void_p * self.L)(*[ctypes.c_void_p(w.data_ptr()) for w in Ws])
        a, b = ctypes.c_size_t(), ctypes.c_size_t()
        st = self._lib.mlp_pipe_run_host(self._h, ctypes.c_void_p(X.data_ptr()), arr, ctypes.c_void_p(Y.data_ptr()),
                                         _stream_ptr(stream), ctypes.byref(a), ctypes.byref(b))
        _check(st, self._h)
        return a.value, b.value

    def hidden(self, layer: int = 1) -> torch.Tensor:
        """Copy of hidden activation H_layer as a CUDA bf16 tensor [M x N_layer] (test hook)."""
        p, n = ctypes.c_void_p(), ctypes.c_size_t()
        _check(self._lib.mlp_pipe_hidden(self._h, layer, ctypes.byref(p), ctypes.byref(n)), self._h)
        out = torch.empty((self.M, self.widths[layer]), dtype=torch.bfloat16, device="cuda")
        assert out.numel() * 2 == n.value
        torch.cuda.synchronize()
        # device-to-device copy through torch: wrap the raw pointer without taking ownership
        src = _RawCudaBuffer(p.value, n.value)
        out.view(torch.uint8).view(-1).copy_(torch.as_tensor(src, device="cuda"))
        return out

    def poison_hidden(self, pattern: int = 0x7FC0, stream: Optional[torch.cuda.Stream] = None):
        _check(self._lib.mlp_pipe_poison_hidden(self._h, pattern, _stream_ptr(stream)), self._h)

    def stats(self) -> mlp_stats:
        s = mlp_stats()
        _check(self._lib.mlp_pipe_stats(self._h, ctypes.byref(s), ctypes.sizeof(s)), self._h)
        return s

    def cta_records(self, cls: int = 0, max_records: int = 256):
        arr = (mlp_cta_record * max_records)()
        n = ctypes.c_int()
        _check(self._lib.mlp_pipe_cta_records(self._h, cls, arr, max_records, ctypes.byref(n)), self._h)
        return [arr[i] for i in range(n.value)]

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.mlp_pipe_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class _RawCudaBuffer:
    """Exposes a raw device pointer through __cuda_array_interface__ (uint8, no ownership)."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def run_static(X: torch.Tensor, Ws: Sequence[torch.Tensor], act: int, Y: Optional[torch.Tensor] = None,
               stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """mlp_pipe_run_static: the CTA-pipelined pass without a handle, for callers that must not allocate device memory.

    The library side allocates nothing: its scratch is a fixed MLP_STATIC_SCRATCH_BYTES array inside the library, shared
    by every call on the device (so calls must not overlap on the GPU; see include/mlp_pipe.h).  Pass `Y` to keep this
    wrapper from allocating the output tensor through torch.
    """
    if not torch.cuda.is_available():
        raise RuntimeError("mlp_pipe needs a CUDA device (sm_100a); there is no CPU fallback")
    lib = load()
    M, widths = int(X.shape[0]), [int(X.shape[1])] + [int(w.shape[0]) for w in Ws]
    L = len(Ws)
    if Y is None:
        Y = torch.empty((M, widths[-1]), dtype=torch.bfloat16, device=X.device)
    xp = _dev_ptr(X, (M, widths[0]), "X")
    yp = _dev_ptr(Y, (M, widths[-1]), "Y")
    wp = (ctypes.c_void_p * L)(*[_dev_ptr(w, (widths[l + 1], widths[l]), f"W[{l}]") for l, w in enumerate(Ws)])
    wd = (ctypes.c_int * (L + 1))(*widths)
    _check(lib.mlp_pipe_run_static(M, L, wd, int(act), xp, wp, yp, _stream_ptr(stream)), None)
    return Y


def plan(M: int, widths: Sequence[int], mode: Optional[mlp_mode] = None, num_sms: int = 148):
    """Host-only: the launch plan for this problem (no device needed).  Returns (mlp_plan, [units of layer 0, ...])."""
    lib = load()
    L = len(widths) - 1
    w = (ctypes.c_int * (L + 1))(*[int(x) for x in widths])
    mp = ctypes.byref(mode) if mode is not None else None
    out = mlp_plan()
    _check(lib.mlp_pipe_plan(int(M), L, w, mp, int(num_sms), ctypes.byref(out)))
    tables = []
    for l in range(L):
        n = ctypes.c_int()
        arr = (mlp_unit * out.units[l])()
        _check(lib.mlp_pipe_plan_units(int(M), L, w, mp, int(num_sms), l, arr, out.units[l], ctypes.byref(n)))
        tables.append([(u.tile, u.kind, u.k_slice, u.begin, u.end) for u in arr])
    return out, tables


def version() -> str:
    return load().mlp_pipe_version().decode()

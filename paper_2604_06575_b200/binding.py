"""Thin ctypes binding of include/polylab.h -- argument marshalling only.

Every step of the path (bounds, pack, expand, sort, segmented sum, prune, unpack) runs in the CUDA
kernels of libpolylab.so; this module turns torch tensors into pointers and sizes, owns nothing but a
cached workspace buffer, and raises PolylabError when the library is missing or a call fails.  There is
no CPU fallback.  torch is used for device memory and streams only.

Function names follow the C ABI: simplify, mul_simplify, expand, pack_keys, simplify_host,
mul_simplify_host (Table 3, Table 4 for the operations themselves).
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpolylab.so")

(OK, ERR_INVALID_ARGUMENT, ERR_KEY_TOO_WIDE, ERR_EXPONENT_RANGE, ERR_WORKSPACE_TOO_SMALL, ERR_OUTPUT_TOO_SMALL, ERR_CUDA,
 ERR_INTERNAL, ERR_RETRY) = range(9)
FLAG_DEVICE_COUNT = 1
FLAG_TIMING = 2
FLAG_SAFE_RANK = 4
FLAG_NO_BUCKET = 8
FLAG_NO_FUSED_PACK = 16
FLAG_EXACT_BOUNDS = 32
FLAG_NO_TABLE = 64
FLAG_NO_SMALL = 128
FLAG_EXACT_HIST = 256
FLAG_NO_GROUP_FINISH = 512
FLAG_DEBUG_GROUP_HANDS_ON = 0x04000000
FLAG_DEBUG_FORCE_TABLE = 0x10000000
FLAG_DEBUG_FORCE_HASH = 0x08000000
FLAG_DEBUG_FORCE_BUCKET = 0x20000000
FLAG_DEBUG_UNSTABLE = 0x40000000
FLAG_DEBUG_NFAST_SHIFT = 16
STAGES = ("bounds", "pack", "sort", "reduce", "prune")
MAX_NVARS = 256
MAX_TERMS = 1 << 30
SMALL_WORKSPACE_BYTES = 65536
STATIC_MAX_TERMS = 65536            # polylab_simplify_static: the library's static workspace holds this many terms
STATIC_WORKSPACE_BYTES = 8 << 20


class PolylabError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"polylab status {status}: {message}")
        self.status = status


class _Stats(ctypes.Structure):
    _fields_ = [("key_bits", ctypes.c_int32), ("key_bytes", ctypes.c_int32), ("sort_passes", ctypes.c_int32),
                ("digit_bits", ctypes.c_int32 * 32), ("sort_terms", ctypes.c_int64), ("distinct", ctypes.c_int64),
                ("survivors", ctypes.c_int64), ("kernel_launches", ctypes.c_int32), ("rank_fallback", ctypes.c_int32),
                ("stage_ms", ctypes.c_float * 8), ("prefix_passes", ctypes.c_int32), ("bucket_fallback", ctypes.c_int32),
                ("refinish_tiles", ctypes.c_int32), ("plan_digits", ctypes.c_int32), ("bounds_sampled", ctypes.c_int32),
                ("bounds_retry", ctypes.c_int32), ("table_path", ctypes.c_int32), ("table_fallback", ctypes.c_int32),
                ("small_path", ctypes.c_int32), ("hist_sampled", ctypes.c_int32), ("hist_retry", ctypes.c_int32), ("grouped_tiles", ctypes.c_int32)]


class _Opts(ctypes.Structure):
    _fields_ = [("exp_type", ctypes.c_int32), ("flags", ctypes.c_uint32), ("term_stride", ctypes.c_int64),
                ("var_stride", ctypes.c_int64), ("max_exp_host", ctypes.POINTER(ctypes.c_uint32)),
                ("status_device", ctypes.c_void_p), ("stats", ctypes.POINTER(_Stats)), ("coef_type", ctypes.c_int32)]


class _Batch(ctypes.Structure):
    _fields_ = [("coef", ctypes.c_void_p), ("exps", ctypes.c_void_p), ("offsets_host", ctypes.POINTER(ctypes.c_int64)),
                ("nentries", ctypes.c_int64), ("nvars", ctypes.c_int32)]


class _Poly(ctypes.Structure):
    _fields_ = [("coef", ctypes.c_void_p), ("exps", ctypes.c_void_p), ("nterms", ctypes.c_int64), ("nvars", ctypes.c_int32)]


@dataclass
class Stats:
    key_bits: int
    key_bytes: int
    sort_passes: int
    digit_bits: list
    sort_terms: int
    distinct: int
    survivors: int
    kernel_launches: int
    stage_ms: dict
    rank_fallback: int = 0
    prefix_passes: int = 0
    bucket_fallback: int = 0
    refinish_tiles: int = 0
    bounds_sampled: int = 0
    bounds_retry: int = 0
    table_path: int = 0
    table_fallback: int = 0
    small_path: int = 0
    hist_sampled: int = 0
    hist_retry: int = 0
    grouped_tiles: int = 0


_lib = None


def lib():
    """The loaded C-ABI library; raises (never falls back) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PolylabError(-1, f"{LIB_PATH} is missing: build it with `python -m paper_2604_06575_b200.build` "
                                   "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i32, dbl, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_size_t
        po, pp = ctypes.POINTER(_Opts), ctypes.POINTER(_Poly)
        L.polylab_simplify_workspace_bytes.argtypes = [i64, i32, po]
        L.polylab_simplify_workspace_bytes.restype = sz
        L.polylab_mul_simplify_workspace_bytes.argtypes = [i64, i64, i32, po]
        L.polylab_mul_simplify_workspace_bytes.restype = sz
        L.polylab_simplify_host_workspace_bytes.argtypes = [i64, i32, po]
        L.polylab_simplify_host_workspace_bytes.restype = sz
        L.polylab_mul_simplify_host_workspace_bytes.argtypes = [i64, i64, i32, po]
        L.polylab_mul_simplify_host_workspace_bytes.restype = sz
        simp = [vp, vp, i64, i32, dbl, po, vp, vp, i64, vp, vp, sz, vp]
        L.polylab_simplify.argtypes = simp
        L.polylab_simplify_host.argtypes = simp
        L.polylab_simplify_static.argtypes = [vp, vp, i64, i32, dbl, po, vp, vp, i64, vp, vp]
        mul = [pp, pp, dbl, po, vp, vp, i64, vp, vp, sz, vp]
        L.polylab_mul_simplify.argtypes = mul
        L.polylab_mul_simplify_host.argtypes = mul
        L.polylab_pow_simplify_workspace_bytes.argtypes = [i64, i32, i32, i64, po]
        L.polylab_pow_simplify_workspace_bytes.restype = sz
        L.polylab_pow_simplify.argtypes = [pp, i32, dbl, po, vp, vp, i64, vp, vp, sz, vp]
        pb = ctypes.POINTER(_Batch)
        L.polylab_simplify_batched_workspace_bytes.argtypes = [i64, i64, i32, po]
        L.polylab_simplify_batched_workspace_bytes.restype = sz
        L.polylab_simplify_batched.argtypes = [pb, dbl, po, vp, vp, i64, vp, vp, sz, vp]
        L.polylab_simplify_batched.restype = ctypes.c_int
        L.polylab_matmul_simplify_workspace_bytes.argtypes = [i64, i64, i64, i64, i64, i64, i32, po]
        L.polylab_matmul_simplify_workspace_bytes.restype = sz
        L.polylab_matmul_simplify.argtypes = [pb, i32, i32, pb, i32, dbl, po, vp, vp, i64, vp, vp, sz, vp]
        L.polylab_matmul_simplify.restype = ctypes.c_int
        L.polylab_expand.argtypes = [pp, pp, po, vp, vp, vp, sz, vp]
        L.polylab_pack_keys.argtypes = [vp, i64, i32, po, vp, ctypes.POINTER(i32), vp, sz, vp]
        for name in ("polylab_simplify", "polylab_simplify_host", "polylab_mul_simplify", "polylab_mul_simplify_host",
                     "polylab_expand", "polylab_pack_keys", "polylab_version", "polylab_pow_simplify"):
            getattr(L, name).restype = ctypes.c_int
        L.polylab_status_string.argtypes = [ctypes.c_int]
        L.polylab_status_string.restype = ctypes.c_char_p
        L.polylab_last_cuda_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(status: int, allow=()):
    if status != OK and status not in allow:
        L = lib()
        msg = L.polylab_status_string(status).decode()
        if status == ERR_CUDA:
            msg += " (" + L.polylab_last_cuda_error().decode() + ")"
        raise PolylabError(status, msg)
    return status


_EXP_TYPE = {torch.uint8: 1, torch.uint16: 2, torch.uint32: 4}
_NP_EXP_TYPE = {np.dtype(np.uint8): 1, np.dtype(np.uint16): 2, np.dtype(np.uint32): 4}
_TORCH_OF_BYTES = {1: torch.uint8, 2: torch.uint16, 4: torch.uint32}


class Workspace:
    """A grow-only device byte buffer reused between calls (the library itself allocates nothing)."""

    def __init__(self, device="cuda"):
        self.device = torch.device(device)
        self.buf: Optional[torch.Tensor] = None

    def get(self, nbytes: int) -> torch.Tensor:
        if self.buf is None or self.buf.numel() < nbytes:
            self.buf = None
            self.buf = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
        return self.buf


_default_ws: dict = {}


def _ws(device, workspace: Optional[Workspace]) -> Workspace:
    if workspace is not None:
        return workspace
    key = str(device)
    if key not in _default_ws:
        _default_ws[key] = Workspace(device)
    return _default_ws[key]


def _stream_ptr(stream) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


_COEF_TYPE = {torch.float64: 0, torch.float32: 1}      # polylab_coef_type


def _make_opts(exp_bytes: int, max_exp, flags: int = 0, strides=None, status_device=None, keep=None, coef_dtype=torch.float64):
    o = _Opts()
    o.exp_type = exp_bytes
    o.coef_type = _COEF_TYPE[coef_dtype]
    o.flags = flags
    if strides is not None:
        o.term_stride, o.var_stride = int(strides[0]), int(strides[1])
    st = _Stats()
    o.stats = ctypes.pointer(st)
    if max_exp is not None:
        arr = np.ascontiguousarray(np.asarray(max_exp, dtype=np.uint32))
        keep.append(arr)
        o.max_exp_host = arr.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32))
    if status_device is not None:
        o.status_device = status_device.data_ptr()
    return o, st


def _stats(st: _Stats) -> Stats:
    return Stats(st.key_bits, st.key_bytes, st.sort_passes, list(st.digit_bits)[:st.plan_digits], st.sort_terms,
                 st.distinct, st.survivors, st.kernel_launches, {k: float(st.stage_ms[i]) for i, k in enumerate(STAGES)},
                 rank_fallback=st.rank_fallback, prefix_passes=st.prefix_passes, bucket_fallback=st.bucket_fallback,
                 refinish_tiles=st.refinish_tiles, bounds_sampled=st.bounds_sampled, bounds_retry=st.bounds_retry,
                 table_path=st.table_path, table_fallback=st.table_fallback, small_path=st.small_path, hist_sampled=st.hist_sampled, hist_retry=st.hist_retry, grouped_tiles=st.grouped_tiles)


def _dev_poly(coef: torch.Tensor, exps: torch.Tensor, strides=None):
    if not (coef.is_cuda and exps.is_cuda):
        raise PolylabError(ERR_INVALID_ARGUMENT, "coef and exps must be CUDA tensors (use simplify_host for host data)")
    if coef.dtype not in _COEF_TYPE or exps.dtype not in _EXP_TYPE:
        raise PolylabError(ERR_INVALID_ARGUMENT, "coef must be float64 (or float32: single-precision storage), exps uint8/uint16/uint32")
    if exps.dim() != 2 or coef.dim() != 1:
        raise PolylabError(ERR_INVALID_ARGUMENT, "coef [nterms], exps [nterms, nvars] (PAPER.md:80)")
    if strides is None:
        if not exps.is_contiguous():
            strides = (exps.stride(0), exps.stride(1))
    if not coef.is_contiguous():
        coef = coef.contiguous()
    if exps.shape[0] != coef.shape[0]:
        raise PolylabError(ERR_INVALID_ARGUMENT, "coefficient vector and exponent matrix need a matching monomial count")
    return coef, exps, strides


def simplify_workspace_bytes(nterms: int, nvars: int) -> int:
    return int(lib().polylab_simplify_workspace_bytes(nterms, nvars, None))


def mul_simplify_workspace_bytes(na: int, nb: int, nvars: int) -> int:
    return int(lib().polylab_mul_simplify_workspace_bytes(na, nb, nvars, None))


def simplify(coef: torch.Tensor, exps: torch.Tensor, tol: float = 0.0, *, max_exp: Optional[Sequence[int]] = None,
             out_capacity: Optional[int] = None, workspace: Optional[Workspace] = None, stream=None,
             out: Optional[tuple] = None, return_stats: bool = False, timing: bool = False, flags: int = 0):
    """polylab_simplify on device tensors: returns (coef[U'], exps[U', nvars]) views of the output buffers.
    `flags`: extra POLYLAB_FLAG_* bits (FLAG_SAFE_RANK, FLAG_DEBUG_UNSTABLE)."""
    coef, exps, strides = _dev_poly(coef, exps)
    n, nvars = int(exps.shape[0]), int(exps.shape[1])
    eb = _EXP_TYPE[exps.dtype]
    cap = n if out_capacity is None else int(out_capacity)
    keep = []
    o, st = _make_opts(eb, max_exp, flags=(FLAG_TIMING if timing else 0) | flags, strides=strides, keep=keep, coef_dtype=coef.dtype)
    if out is None:
        out_coef = torch.empty(max(cap, 1), dtype=coef.dtype, device=coef.device)
        out_exps = torch.empty((max(cap, 1), nvars), dtype=exps.dtype, device=coef.device)
    else:
        out_coef, out_exps = out
    wsb = simplify_workspace_bytes(n, nvars)
    ws = _ws(coef.device, workspace).get(max(wsb, 256))
    count = ctypes.c_int64(0)
    with torch.cuda.device(coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_simplify(coef.data_ptr(), exps.data_ptr(), n, nvars, float(tol), ctypes.byref(o),
                                    out_coef.data_ptr(), out_exps.data_ptr(), cap, ctypes.addressof(count),
                                    ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    k = count.value
    res = (out_coef[:k], out_exps[:k])
    return (*res, _stats(st)) if return_stats else res


def simplify_static(coef: torch.Tensor, exps: torch.Tensor, tol: float = 0.0, *, max_exp: Optional[Sequence[int]] = None,
                    out: Optional[tuple] = None, stream=None, return_stats: bool = False, flags: int = 0):
    """polylab_simplify_static: the same operation with the library's own static device workspace -- no workspace tensor, no
    allocation inside the call; at most STATIC_MAX_TERMS terms (ERR_WORKSPACE_TOO_SMALL beyond).  `out` = (out_coef, out_exps)
    buffers of the caller (allocated here when omitted: the C entry point itself allocates nothing).  Calls share one
    array per GPU: do not overlap them."""
    coef, exps, strides = _dev_poly(coef, exps)
    n, nvars = int(exps.shape[0]), int(exps.shape[1])
    keep = []
    o, st = _make_opts(_EXP_TYPE[exps.dtype], max_exp, flags=flags, strides=strides, keep=keep, coef_dtype=coef.dtype)
    if out is None:
        out_coef = torch.empty(max(n, 1), dtype=coef.dtype, device=coef.device)
        out_exps = torch.empty((max(n, 1), nvars), dtype=exps.dtype, device=coef.device)
    else:
        out_coef, out_exps = out
    count = ctypes.c_int64(0)
    with torch.cuda.device(coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_simplify_static(coef.data_ptr(), exps.data_ptr(), n, nvars, float(tol), ctypes.byref(o),
                                           out_coef.data_ptr(), out_exps.data_ptr(), int(out_coef.shape[0]),
                                           ctypes.addressof(count), _stream_ptr(stream))
    _check(rc)
    k = count.value
    res = (out_coef[:k], out_exps[:k])
    return (*res, _stats(st)) if return_stats else res


def simplify_async(coef: torch.Tensor, exps: torch.Tensor, tol: float, max_exp: Sequence[int], out_coef: torch.Tensor,
                   out_exps: torch.Tensor, out_count: torch.Tensor, status: Optional[torch.Tensor],
                   workspace: Optional[Workspace] = None, stream=None, flags: int = 0) -> Stats:
    """polylab_simplify with POLYLAB_FLAG_DEVICE_COUNT: no host synchronisation; count/status stay on the device.
    `status` may come back as ERR_RETRY (a self-check of the fast path failed): call again with
    flags=FLAG_SAFE_RANK | FLAG_NO_BUCKET."""
    coef, exps, strides = _dev_poly(coef, exps)
    n, nvars = int(exps.shape[0]), int(exps.shape[1])
    keep = []
    o, st = _make_opts(_EXP_TYPE[exps.dtype], max_exp, flags=FLAG_DEVICE_COUNT | flags, strides=strides, status_device=status, keep=keep,
                       coef_dtype=coef.dtype)
    wsb = simplify_workspace_bytes(n, nvars)
    ws = _ws(coef.device, workspace).get(max(wsb, 256))
    with torch.cuda.device(coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_simplify(coef.data_ptr(), exps.data_ptr(), n, nvars, float(tol), ctypes.byref(o),
                                    out_coef.data_ptr(), out_exps.data_ptr(), int(out_coef.shape[0]), out_count.data_ptr(),
                                    ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    return _stats(st)


def mul_simplify(a_coef: torch.Tensor, a_exps: torch.Tensor, b_coef: torch.Tensor, b_exps: torch.Tensor, tol: float = 0.0, *,
                 max_exp: Optional[Sequence[int]] = None, out_capacity: Optional[int] = None,
                 workspace: Optional[Workspace] = None, stream=None, return_stats: bool = False, timing: bool = False,
                 flags: int = 0):
    """polylab_mul_simplify on device tensors: simplify(a*b)."""
    a_coef, a_exps, sa = _dev_poly(a_coef, a_exps)
    b_coef, b_exps, sb = _dev_poly(b_coef, b_exps)
    if sa is not None or sb is not None:
        a_exps, b_exps = a_exps.contiguous(), b_exps.contiguous()
    if a_exps.dtype != b_exps.dtype or a_exps.shape[1] != b_exps.shape[1] or a_coef.dtype != b_coef.dtype:
        raise PolylabError(ERR_INVALID_ARGUMENT, "operands must share dtypes and variable space (PAPER.md:175)")
    na, nb, nvars = int(a_exps.shape[0]), int(b_exps.shape[0]), int(a_exps.shape[1])
    n = na * nb
    if n >= MAX_TERMS:
        raise PolylabError(ERR_INVALID_ARGUMENT, "na*nb must be < 2^30")
    cap = n if out_capacity is None else int(out_capacity)
    keep = []
    o, st = _make_opts(_EXP_TYPE[a_exps.dtype], max_exp, flags=(FLAG_TIMING if timing else 0) | flags, keep=keep, coef_dtype=a_coef.dtype)
    out_coef = torch.empty(max(cap, 1), dtype=a_coef.dtype, device=a_coef.device)
    out_exps = torch.empty((max(cap, 1), nvars), dtype=a_exps.dtype, device=a_coef.device)
    wsb = mul_simplify_workspace_bytes(na, nb, nvars)
    ws = _ws(a_coef.device, workspace).get(max(wsb, 256))
    pa = _Poly(a_coef.data_ptr(), a_exps.data_ptr(), na, nvars)
    pb = _Poly(b_coef.data_ptr(), b_exps.data_ptr(), nb, nvars)
    count = ctypes.c_int64(0)
    with torch.cuda.device(a_coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_mul_simplify(ctypes.byref(pa), ctypes.byref(pb), float(tol), ctypes.byref(o), out_coef.data_ptr(),
                                        out_exps.data_ptr(), cap, ctypes.addressof(count), ws.data_ptr(), ws.numel(),
                                        _stream_ptr(stream))
    _check(rc)
    k = count.value
    res = (out_coef[:k], out_exps[:k])
    return (*res, _stats(st)) if return_stats else res


def pow_simplify(coef: torch.Tensor, exps: torch.Tensor, power: int, tol: float = 0.0, *, out_capacity: Optional[int] = None,
                 workspace: Optional[Workspace] = None, stream=None, return_stats: bool = False, flags: int = 0):
    """polylab_pow_simplify on device tensors: simplify(p^power); the intermediate powers stay inside the workspace.
    out_capacity bounds every power's term count (default: min(nterms^power, 2^22))."""
    coef, exps, strides = _dev_poly(coef, exps)
    if strides is not None:
        exps = exps.contiguous()
    n, nvars = int(exps.shape[0]), int(exps.shape[1])
    cap = int(out_capacity) if out_capacity is not None else max(1, min(max(n, 1) ** max(int(power), 1), 1 << 22))
    keep = []
    o, st = _make_opts(_EXP_TYPE[exps.dtype], None, flags=flags, keep=keep, coef_dtype=coef.dtype)
    out_coef = torch.empty(max(cap, 1), dtype=coef.dtype, device=coef.device)
    out_exps = torch.empty((max(cap, 1), nvars), dtype=exps.dtype, device=coef.device)
    wsb = int(lib().polylab_pow_simplify_workspace_bytes(n, nvars, int(power), cap, ctypes.byref(o)))
    if wsb == 0 and n > 0 and power > 1:
        raise PolylabError(ERR_INVALID_ARGUMENT, "out_capacity * nterms must be < 2^30")
    ws = _ws(coef.device, workspace).get(max(wsb, 256))
    pp = _Poly(coef.data_ptr(), exps.data_ptr(), n, nvars)
    count = ctypes.c_int64(0)
    with torch.cuda.device(coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_pow_simplify(ctypes.byref(pp), int(power), float(tol), ctypes.byref(o), out_coef.data_ptr(),
                                        out_exps.data_ptr(), cap, ctypes.addressof(count), ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    k = count.value
    res = (out_coef[:k], out_exps[:k])
    return (*res, _stats(st)) if return_stats else res


def _batch(coef: torch.Tensor, exps: torch.Tensor, offsets, keep: list):
    coef, exps, strides = _dev_poly(coef, exps)
    if strides is not None:
        exps = exps.contiguous()
    off = np.ascontiguousarray(np.asarray(offsets, dtype=np.int64))
    if off.ndim != 1 or off.shape[0] < 1 or int(off[-1]) != int(coef.shape[0]):
        raise PolylabError(ERR_INVALID_ARGUMENT, "offsets must be a 1-D array of nentries + 1 values ending at the term count")
    keep.extend([coef, exps, off])
    return _Batch(coef.data_ptr(), exps.data_ptr(), off.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), off.shape[0] - 1,
                  int(exps.shape[1])), coef, exps, off


def simplify_batched(coef: torch.Tensor, exps: torch.Tensor, offsets, tol: float = 0.0, *, out_capacity: Optional[int] = None,
                     workspace: Optional[Workspace] = None, stream=None, return_stats: bool = False, flags: int = 0):
    """polylab_simplify_batched: entry e = terms [offsets[e], offsets[e+1]); returns (coef, exps, out_offsets) with the
    simplified entries concatenated in entry order (polynomial matrices, sum)."""
    keep = []
    bt, coef, exps, off = _batch(coef, exps, offsets, keep)
    n, ne, nvars = int(coef.shape[0]), int(off.shape[0] - 1), int(exps.shape[1])
    cap = n if out_capacity is None else int(out_capacity)
    o, st = _make_opts(_EXP_TYPE[exps.dtype], None, flags=flags, keep=keep, coef_dtype=coef.dtype)
    out_coef = torch.empty(max(cap, 1), dtype=coef.dtype, device=coef.device)
    out_exps = torch.empty((max(cap, 1), nvars), dtype=exps.dtype, device=coef.device)
    out_off = np.zeros(ne + 1, dtype=np.int64)
    wsb = int(lib().polylab_simplify_batched_workspace_bytes(n, ne, nvars, ctypes.byref(o)))
    ws = _ws(coef.device, workspace).get(max(wsb, 256))
    with torch.cuda.device(coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_simplify_batched(ctypes.byref(bt), float(tol), ctypes.byref(o), out_coef.data_ptr(), out_exps.data_ptr(), cap,
                                            out_off.ctypes.data, ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    k = int(out_off[-1])
    res = (out_coef[:k], out_exps[:k], out_off)
    return (*res, _stats(st)) if return_stats else res


def matmul_simplify(a_coef: torch.Tensor, a_exps: torch.Tensor, a_offsets, b_coef: torch.Tensor, b_exps: torch.Tensor, b_offsets,
                    m: int, k: int, n: int, tol: float = 0.0, *, out_capacity: Optional[int] = None,
                    workspace: Optional[Workspace] = None, stream=None, return_stats: bool = False, flags: int = 0):
    """polylab_matmul_simplify: simplify(A*B) for polynomial matrices A (m x k) and B (k x n) given as row-major batches;
    returns (coef, exps, out_offsets) of the m*n entries (Table 4)."""
    keep = []
    ba, a_coef, a_exps, aoff = _batch(a_coef, a_exps, a_offsets, keep)
    bb, b_coef, b_exps, boff = _batch(b_coef, b_exps, b_offsets, keep)
    if a_exps.dtype != b_exps.dtype or a_exps.shape[1] != b_exps.shape[1] or a_coef.dtype != b_coef.dtype:
        raise PolylabError(ERR_INVALID_ARGUMENT, "operands must share dtypes and variable space (PAPER.md:175)")
    if aoff.shape[0] - 1 != m * k or boff.shape[0] - 1 != k * n:
        raise PolylabError(ERR_INVALID_ARGUMENT, "A needs m*k entries and B k*n entries (row-major)")
    na_e, nb_e = np.diff(aoff).reshape(m, k), np.diff(boff).reshape(k, n)
    nprod = int((na_e.astype(np.int64) @ nb_e.astype(np.int64)).sum())
    nvars = int(a_exps.shape[1])
    cap = nprod if out_capacity is None else int(out_capacity)
    o, st = _make_opts(_EXP_TYPE[a_exps.dtype], None, flags=flags, keep=keep, coef_dtype=a_coef.dtype)
    out_coef = torch.empty(max(cap, 1), dtype=a_coef.dtype, device=a_coef.device)
    out_exps = torch.empty((max(cap, 1), nvars), dtype=a_exps.dtype, device=a_coef.device)
    out_off = np.zeros(m * n + 1, dtype=np.int64)
    wsb = int(lib().polylab_matmul_simplify_workspace_bytes(nprod, int(aoff[-1]), int(boff[-1]), m, k, n, nvars, ctypes.byref(o)))
    if wsb == 0:
        raise PolylabError(ERR_INVALID_ARGUMENT, "the matrix product has 2^30 or more term products")
    ws = _ws(a_coef.device, workspace).get(max(wsb, 256))
    with torch.cuda.device(a_coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_matmul_simplify(ctypes.byref(ba), m, k, ctypes.byref(bb), n, float(tol), ctypes.byref(o), out_coef.data_ptr(),
                                           out_exps.data_ptr(), cap, out_off.ctypes.data, ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    kk = int(out_off[-1])
    res = (out_coef[:kk], out_exps[:kk], out_off)
    return (*res, _stats(st)) if return_stats else res


def expand(a_coef: torch.Tensor, a_exps: torch.Tensor, b_coef: torch.Tensor, b_exps: torch.Tensor, stream=None):
    """polylab_expand: the raw product, term (i,j) at i*nb+j, not merged."""
    a_coef, a_exps, _ = _dev_poly(a_coef, a_exps.contiguous())
    b_coef, b_exps, _ = _dev_poly(b_coef, b_exps.contiguous())
    na, nb, nvars = int(a_exps.shape[0]), int(b_exps.shape[0]), int(a_exps.shape[1])
    n = na * nb
    keep = []
    if a_coef.dtype != b_coef.dtype:
        raise PolylabError(ERR_INVALID_ARGUMENT, "operands must share the coefficient dtype")
    o, _ = _make_opts(_EXP_TYPE[a_exps.dtype], None, keep=keep, coef_dtype=a_coef.dtype)
    out_coef = torch.empty(max(n, 1), dtype=a_coef.dtype, device=a_coef.device)
    out_exps = torch.empty((max(n, 1), nvars), dtype=a_exps.dtype, device=a_coef.device)
    ws = torch.empty(SMALL_WORKSPACE_BYTES, dtype=torch.uint8, device=a_coef.device)
    pa = _Poly(a_coef.data_ptr(), a_exps.data_ptr(), na, nvars)
    pb = _Poly(b_coef.data_ptr(), b_exps.data_ptr(), nb, nvars)
    with torch.cuda.device(a_coef.device):     # the library launches on the CURRENT device
        rc = lib().polylab_expand(ctypes.byref(pa), ctypes.byref(pb), ctypes.byref(o), out_coef.data_ptr(), out_exps.data_ptr(),
                                  ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    return out_coef[:n], out_exps[:n]


def pack_keys(exps: torch.Tensor, max_exp: Optional[Sequence[int]] = None, stream=None):
    """polylab_pack_keys: (keys [nterms, 2] uint64 as (hi, lo) -- returned as int64 bit patterns --, key_bits)."""
    if not exps.is_cuda or exps.dtype not in _EXP_TYPE or exps.dim() != 2:
        raise PolylabError(ERR_INVALID_ARGUMENT, "exps must be a 2-D CUDA tensor of uint8/uint16/uint32")
    strides = None if exps.is_contiguous() else (exps.stride(0), exps.stride(1))
    n, nvars = int(exps.shape[0]), int(exps.shape[1])
    keep = []
    o, _ = _make_opts(_EXP_TYPE[exps.dtype], max_exp, strides=strides, keep=keep)
    out = torch.zeros((max(n, 1), 2), dtype=torch.int64, device=exps.device)
    ws = torch.empty(SMALL_WORKSPACE_BYTES, dtype=torch.uint8, device=exps.device)
    bits = ctypes.c_int32(0)
    with torch.cuda.device(exps.device):     # the library launches on the CURRENT device
        rc = lib().polylab_pack_keys(exps.data_ptr(), n, nvars, ctypes.byref(o), out.data_ptr(), ctypes.byref(bits),
                                     ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    return out[:n], bits.value


# ---------------------------------------------------------------------------- host-buffer calls

def _host_arrays(coef, exps):
    coef = np.ascontiguousarray(coef, dtype=np.float64).reshape(-1) if not isinstance(coef, torch.Tensor) else coef
    if isinstance(coef, torch.Tensor):
        cptr, n = coef.data_ptr(), int(coef.shape[0])
    else:
        cptr, n = coef.ctypes.data, int(coef.shape[0])
    if isinstance(exps, torch.Tensor):
        eb, eptr, nvars = _EXP_TYPE[exps.dtype], exps.data_ptr(), int(exps.shape[1])
        if not exps.is_contiguous():
            raise PolylabError(ERR_INVALID_ARGUMENT, "host exps must be contiguous")
    else:
        exps = np.ascontiguousarray(exps)
        if exps.dtype not in _NP_EXP_TYPE:
            raise PolylabError(ERR_INVALID_ARGUMENT, "host exps must be uint8/uint16/uint32")
        eb, eptr, nvars = _NP_EXP_TYPE[exps.dtype], exps.ctypes.data, int(exps.shape[1])
    if int(exps.shape[0]) != n:
        raise PolylabError(ERR_INVALID_ARGUMENT, "coefficient vector and exponent matrix need a matching monomial count")
    return (coef, exps), cptr, eptr, n, nvars, eb


def simplify_host(coef, exps, tol: float = 0.0, *, max_exp=None, out: Optional[tuple] = None,
                  workspace: Optional[Workspace] = None, device="cuda", stream=None, return_stats: bool = False):
    """polylab_simplify_host: numpy arrays or (pinned) CPU tensors in, numpy arrays (or the given `out` CPU tensors) out.
    Host<->device copies happen inside the C call."""
    keepalive, cptr, eptr, n, nvars, eb = _host_arrays(coef, exps)
    keep = []
    o, st = _make_opts(eb, max_exp, keep=keep)
    if out is None:
        out_coef = torch.empty(max(n, 1), dtype=torch.float64)
        out_exps = torch.empty((max(n, 1), nvars), dtype=_TORCH_OF_BYTES[eb])
    else:
        out_coef, out_exps = out
    wsb = int(lib().polylab_simplify_host_workspace_bytes(n, nvars, ctypes.byref(o)))
    ws = _ws(torch.device(device), workspace).get(max(wsb, 256))
    count = ctypes.c_int64(0)
    with torch.cuda.device(ws.device):
        rc = lib().polylab_simplify_host(cptr, eptr, n, nvars, float(tol), ctypes.byref(o), out_coef.data_ptr(),
                                         out_exps.data_ptr(), int(out_coef.shape[0]), ctypes.addressof(count),
                                         ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    k = count.value
    res = (out_coef[:k].numpy(), out_exps[:k].numpy()) if out is None else (out_coef[:k], out_exps[:k])
    return (*res, _stats(st)) if return_stats else res


def mul_simplify_host(a_coef, a_exps, b_coef, b_exps, tol: float = 0.0, *, max_exp=None,
                      workspace: Optional[Workspace] = None, device="cuda", stream=None, return_stats: bool = False):
    """polylab_mul_simplify_host: host operands in, numpy result out; copies inside the C call."""
    ka, ca, ea, na, nvars, eb = _host_arrays(a_coef, a_exps)
    kb, cb, ebp, nb, nvars_b, eb_b = _host_arrays(b_coef, b_exps)
    if nvars != nvars_b or eb != eb_b:
        raise PolylabError(ERR_INVALID_ARGUMENT, "operands must share dtype and variable space (PAPER.md:175)")
    n = na * nb
    keep = []
    o, st = _make_opts(eb, max_exp, keep=keep)
    out_coef = torch.empty(max(n, 1), dtype=torch.float64)
    out_exps = torch.empty((max(n, 1), nvars), dtype=_TORCH_OF_BYTES[eb])
    wsb = int(lib().polylab_mul_simplify_host_workspace_bytes(na, nb, nvars, ctypes.byref(o)))
    ws = _ws(torch.device(device), workspace).get(max(wsb, 256))
    pa, pb = _Poly(ca, ea, na, nvars), _Poly(cb, ebp, nb, nvars)
    count = ctypes.c_int64(0)
    with torch.cuda.device(ws.device):
        rc = lib().polylab_mul_simplify_host(ctypes.byref(pa), ctypes.byref(pb), float(tol), ctypes.byref(o),
                                             out_coef.data_ptr(), out_exps.data_ptr(), n, ctypes.addressof(count),
                                             ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    k = count.value
    res = (out_coef[:k].numpy(), out_exps[:k].numpy())
    return (*res, _stats(st)) if return_stats else res

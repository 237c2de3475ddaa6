"""ctypes front end of the CPU oracle (oracle/polylab_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_2604_06575_b200 and shares no code with the CUDA
path.  All arithmetic of the method lives in the C file; this module only
builds it (gcc), marshals numpy arrays and returns numpy arrays.

Definitions follow PAPER.md:80-81 (Table 3), PAPER.md:117-119 (Table 4); see
polylab_oracle.h for the readings (A1 order, A2 prune predicate, A6 rounding).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "polylab_oracle.c")
_HDR = os.path.join(_HERE, "polylab_oracle.h")
_LIB = os.path.join(_HERE, "libpolylab_oracle.so")

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-ffp-contract=off: products are rounded once)."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        tmp = f"{_LIB}.{os.getpid()}.tmp"     # atomic replace: safe under parallel ranks
        cmd = ["gcc", "-std=c11", "-O2", "-Wall", "-Wextra", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, i32, dbl, vp = ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_void_p
        simp_args = [vp, vp, i32, i64, i32, dbl, vp, vp, vp, vp, vp]
        for name in ("oracle_simplify", "oracle_simplify_sortscan"):
            getattr(lib, name).argtypes = simp_args
            getattr(lib, name).restype = i64
        lib.oracle_expand.argtypes = [vp, vp, i64, vp, vp, i64, i32, i32, vp, vp]
        lib.oracle_expand.restype = i64
        lib.oracle_mul_simplify.argtypes = [vp, vp, i64, vp, vp, i64, i32, i32, dbl, vp, vp, vp, vp, vp]
        lib.oracle_mul_simplify.restype = i64
        lib.oracle_eval.argtypes = [vp, vp, i32, i64, i32, vp, vp, vp]
        lib.oracle_eval.restype = ctypes.c_int
        _lib = lib
    return _lib


@dataclass
class OracleResult:
    """All distinct monomials of the input, UNPRUNED, ascending lexicographic.

    rows[k] is monomial m_k, sum[k] = s_m, abs[k] = A_m = sum of |contributions|,
    count[k] = |I_m|, keep[k] = (|s_m| > tol).
    """
    rows: np.ndarray    # [U, nvars] uint32
    sum: np.ndarray     # [U] float64
    abs: np.ndarray     # [U] float64
    count: np.ndarray   # [U] int64
    keep: np.ndarray    # [U] bool
    tol: float

    @property
    def pruned(self):
        """(coef, rows) of the simplified polynomial: survivors only."""
        return self.sum[self.keep], self.rows[self.keep]


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _prep(coef, exps):
    coef = np.ascontiguousarray(coef, dtype=np.float64).reshape(-1)
    exps = np.ascontiguousarray(exps)
    if exps.dtype not in (np.uint8, np.uint16, np.uint32):
        if np.any(np.asarray(exps) < 0):
            raise ValueError("exponents must be non-negative integers (PAPER.md:165)")
        exps = np.ascontiguousarray(exps, dtype=np.uint32)
    if exps.ndim != 2 or exps.shape[0] != coef.shape[0]:
        raise ValueError("coefficient vector and exponent matrix need a matching monomial count (PAPER.md:80)")
    return coef, exps


def _alloc(n, nvars):
    return (np.zeros((n, nvars), np.uint32), np.zeros(n, np.float64), np.zeros(n, np.float64),
            np.zeros(n, np.int64), np.zeros(n, np.uint8))


def _finish(U, outs, tol):
    if U < 0:
        raise RuntimeError("oracle rejected its arguments or ran out of memory")
    rows, s, a, c, k = outs
    return OracleResult(rows[:U].copy(), s[:U].copy(), a[:U].copy(), c[:U].copy(), k[:U].astype(bool), float(tol))


def simplify(coef, exps, tol: float = 0.0, method: str = "hash") -> OracleResult:
    """simplify(p, zeroprec) of PAPER.md:81/119 on (coef, exps); method 'hash' or 'sortscan'."""
    coef, exps = _prep(coef, exps)
    n, nvars = exps.shape
    if nvars < 1:
        raise ValueError("nvars must be >= 1")
    outs = _alloc(max(n, 1), nvars)
    fn = _load().oracle_simplify if method == "hash" else _load().oracle_simplify_sortscan
    U = fn(_ptr(coef), _ptr(exps), exps.dtype.itemsize, n, nvars, float(tol), *[_ptr(o) for o in outs])
    return _finish(U, outs, tol)


def expand(ca, ea, cb, eb):
    """Raw product terms (coef [na*nb], rows [na*nb, nvars] uint32)."""
    ca, ea = _prep(ca, ea)
    cb, eb = _prep(cb, eb)
    if ea.dtype != eb.dtype or ea.shape[1] != eb.shape[1]:
        raise ValueError("operands must share dtype and variable space (aligned before the op, PAPER.md:175)")
    na, nb, nvars = ea.shape[0], eb.shape[0], ea.shape[1]
    oc = np.zeros(max(na * nb, 1), np.float64)
    orow = np.zeros((max(na * nb, 1), nvars), np.uint32)
    N = _load().oracle_expand(_ptr(ca), _ptr(ea), na, _ptr(cb), _ptr(eb), nb, ea.dtype.itemsize, nvars,
                              _ptr(oc), _ptr(orow))
    if N < 0:
        raise RuntimeError("oracle_expand rejected its arguments")
    return oc[:N].copy(), orow[:N].copy()


def mul_simplify(ca, ea, cb, eb, tol: float = 0.0) -> OracleResult:
    """simplify(a*b): all na*nb term products, then merged."""
    ca, ea = _prep(ca, ea)
    cb, eb = _prep(cb, eb)
    if ea.dtype != eb.dtype or ea.shape[1] != eb.shape[1]:
        raise ValueError("operands must share dtype and variable space (aligned before the op, PAPER.md:175)")
    na, nb, nvars = ea.shape[0], eb.shape[0], ea.shape[1]
    outs = _alloc(max(na * nb, 1), nvars)
    U = _load().oracle_mul_simplify(_ptr(ca), _ptr(ea), na, _ptr(cb), _ptr(eb), nb, ea.dtype.itemsize, nvars,
                                    float(tol), *[_ptr(o) for o in outs])
    return _finish(U, outs, tol)


def evaluate(coef, exps, x):
    """(p(x), sum_t |c_t x^alpha_t|) in long double -- the paper's eval."""
    coef, exps = _prep(coef, exps)
    x = np.ascontiguousarray(x, dtype=np.float64).reshape(-1)
    if x.shape[0] != exps.shape[1]:
        raise ValueError("point dimension must equal nvars")
    val, ab = ctypes.c_double(0.0), ctypes.c_double(0.0)
    rc = _load().oracle_eval(_ptr(coef), _ptr(exps), exps.dtype.itemsize, exps.shape[0], exps.shape[1],
                             _ptr(x), ctypes.byref(val), ctypes.byref(ab))
    if rc != 0:
        raise RuntimeError("oracle_eval rejected its arguments")
    return val.value, ab.value

"""CPU-only checks of the boundary: the library builds, loads, exports every symbol include/polylab.h
declares, and rejects bad arguments on the host before any CUDA work (no compute calls here)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "polylab.h")


@pytest.fixture(scope="module")
def L():
    from paper_2604_06575_b200 import build
    build.build()
    from paper_2604_06575_b200 import binding
    return binding.lib()


def _declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(polylab_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported(L):
    names = _declared_functions()
    assert {"polylab_simplify", "polylab_mul_simplify", "polylab_expand", "polylab_pack_keys", "polylab_simplify_host",
            "polylab_mul_simplify_host", "polylab_simplify_workspace_bytes", "polylab_mul_simplify_workspace_bytes",
            "polylab_status_string", "polylab_version", "polylab_pow_simplify", "polylab_pow_simplify_workspace_bytes",
            "polylab_simplify_batched", "polylab_simplify_batched_workspace_bytes", "polylab_matmul_simplify",
            "polylab_matmul_simplify_workspace_bytes"} <= set(names)
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/polylab.h but not exported"


def test_header_is_plain_c(tmp_path):
    """The header compiles as C99 with no CUDA or C++ in sight."""
    src = tmp_path / "t.c"
    src.write_text('#include "polylab.h"\nint main(void){polylab_opts o = {0}; polylab_stats s = {0}; (void)o; (void)s; return POLYLAB_OK;}\n')
    import subprocess
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src), "-o",
                    str(tmp_path / "t.o")], check=True)


def test_struct_layouts_match(L, tmp_path):
    """ctypes mirrors of polylab_opts / polylab_stats / polylab_poly have the C sizes."""
    from paper_2604_06575_b200 import binding
    src = tmp_path / "s.c"
    src.write_text('#include <stdio.h>\n#include "polylab.h"\nint main(void){printf("%zu %zu %zu\\n", sizeof(polylab_opts), '
                   'sizeof(polylab_stats), sizeof(polylab_poly)); return 0;}\n')
    import subprocess
    exe = tmp_path / "s"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    sizes = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    assert sizes == [ctypes.sizeof(binding._Opts), ctypes.sizeof(binding._Stats), ctypes.sizeof(binding._Poly)]


def test_flag_values_match_the_header(tmp_path):
    """binding.py's FLAG_* constants are the header's POLYLAB_FLAG_* (the fast-digits test hook once shared bit 8 with
    POLYLAB_FLAG_EXACT_HIST: every flag owns its bits)."""
    from paper_2604_06575_b200 import binding
    names = ["DEVICE_COUNT", "TIMING", "SAFE_RANK", "NO_BUCKET", "NO_FUSED_PACK", "EXACT_BOUNDS", "NO_TABLE", "NO_SMALL", "EXACT_HIST",
             "NO_GROUP_FINISH", "DEBUG_FORCE_TABLE", "DEBUG_FORCE_HASH", "DEBUG_FORCE_BUCKET", "DEBUG_UNSTABLE", "DEBUG_GROUP_HANDS_ON"]
    src = tmp_path / "f.c"
    body = "".join('printf("%%u\\n", (unsigned)POLYLAB_FLAG_%s);' % n for n in names)
    src.write_text('#include <stdio.h>\n#include "polylab.h"\nint main(void){%s printf("%%d\\n", POLYLAB_FLAG_DEBUG_NFAST_SHIFT); return 0;}\n' % body)
    import subprocess
    exe = tmp_path / "f"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    vals = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    assert vals[:-1] == [getattr(binding, "FLAG_" + n) for n in names]
    assert vals[-1] == binding.FLAG_DEBUG_NFAST_SHIFT
    used = 0
    for v in vals[:-1] + [0xf << vals[-1]]:
        assert used & v == 0, "two flags share a bit"
        used |= v


def test_version_and_status_strings(L):
    assert L.polylab_version() == 120
    seen = {L.polylab_status_string(i).decode() for i in range(9)}
    assert len(seen) == 9 and "ok" in seen
    assert L.polylab_status_string(99).decode() == "unknown status"


def test_workspace_queries(L):
    small = L.polylab_simplify_workspace_bytes(1000, 4, None)
    big = L.polylab_simplify_workspace_bytes(100_000, 4, None)
    assert 0 < small < big
    # two 16-byte key buffers + two coefficient buffers dominate: 48 B per term (+ 20 B per slot of the table path's
    # dense table, at most max(N, 65536) slots)
    assert 48 * 100_000 <= big <= 68 * 100_000 + (1 << 21)
    assert L.polylab_mul_simplify_workspace_bytes(2000, 2000, 6, None) >= 48 * 4_000_000
    assert L.polylab_mul_simplify_workspace_bytes(1 << 20, 1 << 20, 6, None) == 0      # na*nb >= 2^30
    assert L.polylab_simplify_workspace_bytes(-1, 4, None) == 0
    assert L.polylab_simplify_host_workspace_bytes(1000, 4, None) > small


def test_host_side_argument_errors(L):
    """Argument errors are detected before any launch; none of these touches the GPU."""
    from paper_2604_06575_b200 import binding as B
    cnt = ctypes.c_int64(-7)
    one = ctypes.c_void_p(16)       # never dereferenced: validation fails first
    f = L.polylab_simplify
    args = dict(coef=one, exps=one, n=10, nvars=4, tol=0.0, opts=None, oc=one, oe=one, cap=10, cnt=ctypes.addressof(cnt), ws=one, wsb=1 << 20, st=None)

    def call(**kw):
        a = dict(args, **kw)
        return f(a["coef"], a["exps"], a["n"], a["nvars"], a["tol"], a["opts"], a["oc"], a["oe"], a["cap"], a["cnt"], a["ws"], a["wsb"], a["st"])

    assert call(nvars=0) == B.ERR_INVALID_ARGUMENT
    assert call(nvars=B.MAX_NVARS + 1) == B.ERR_INVALID_ARGUMENT
    assert call(n=-1) == B.ERR_INVALID_ARGUMENT
    assert call(n=B.MAX_TERMS) == B.ERR_INVALID_ARGUMENT
    assert call(tol=float("nan")) == B.ERR_INVALID_ARGUMENT
    assert call(tol=-1.0) == B.ERR_INVALID_ARGUMENT
    assert call(tol=float("inf")) == B.ERR_INVALID_ARGUMENT
    assert call(cnt=None) == B.ERR_INVALID_ARGUMENT
    assert call(coef=None) == B.ERR_INVALID_ARGUMENT
    assert call(ws=None) == B.ERR_INVALID_ARGUMENT
    o = B._Opts()
    o.exp_type = 3
    assert call(opts=ctypes.byref(o)) == B.ERR_INVALID_ARGUMENT
    o = B._Opts()
    o.flags = B.FLAG_DEVICE_COUNT         # device count needs caller bounds
    assert call(opts=ctypes.byref(o)) == B.ERR_INVALID_ARGUMENT
    # nterms == 0 is valid and needs no device: the zero polynomial (reading A3)
    assert call(n=0, coef=None, exps=None, ws=None, wsb=0) == B.OK and cnt.value == 0
    # product: mismatched variable spaces, oversize product
    pa = B._Poly(16, 16, 5, 3)
    pb = B._Poly(16, 16, 5, 4)
    g = L.polylab_mul_simplify
    assert g(ctypes.byref(pa), ctypes.byref(pb), 0.0, None, one, one, 25, ctypes.addressof(cnt), one, 1 << 20, None) == B.ERR_INVALID_ARGUMENT
    pb = B._Poly(16, 16, 1 << 29, 3)
    assert g(ctypes.byref(pa), ctypes.byref(pb), 0.0, None, one, one, 25, ctypes.addressof(cnt), one, 1 << 20, None) == B.ERR_INVALID_ARGUMENT
    pb = B._Poly(None, None, 0, 3)
    cnt.value = -7
    assert g(ctypes.byref(pa), ctypes.byref(pb), 0.0, None, one, one, 25, ctypes.addressof(cnt), one, 1 << 20, None) == B.OK
    assert cnt.value == 0


def test_batched_host_side_checks(L):
    """Batched entry points: argument errors are found on the host (no GPU needed); an all-empty batch returns zero offsets."""
    from paper_2604_06575_b200 import binding as B
    off = (ctypes.c_int64 * 4)(0, 0, 0, 0)
    out_off = (ctypes.c_int64 * 4)(7, 7, 7, 7)
    b = B._Batch(None, None, off, 3, 2)
    assert L.polylab_simplify_batched(ctypes.byref(b), 0.0, None, None, None, 0, out_off, None, 0, None) == B.OK
    assert list(out_off) == [0, 0, 0, 0]
    assert L.polylab_simplify_batched(ctypes.byref(b), -1.0, None, None, None, 0, out_off, None, 0, None) == B.ERR_INVALID_ARGUMENT
    bad = (ctypes.c_int64 * 4)(0, 2, 1, 3)                       # decreasing offsets
    b2 = B._Batch(1, 1, bad, 3, 2)
    assert L.polylab_simplify_batched(ctypes.byref(b2), 0.0, None, None, None, 0, out_off, None, 0, None) == B.ERR_INVALID_ARGUMENT
    b3 = B._Batch(None, None, off, 3, 256)                       # the entry index needs a field of its own: nvars <= 255
    assert L.polylab_simplify_batched(ctypes.byref(b3), 0.0, None, None, None, 0, out_off, None, 0, None) == B.ERR_INVALID_ARGUMENT
    # matrix product: A must have m*k entries, B k*n
    assert L.polylab_matmul_simplify(ctypes.byref(b), 2, 2, ctypes.byref(b), 2, 0.0, None, None, None, 0, out_off, None, 0, None) == B.ERR_INVALID_ARGUMENT
    assert L.polylab_matmul_simplify(ctypes.byref(b), 1, 3, ctypes.byref(b), 1, 0.0, None, None, None, 0, out_off, None, 0, None) == B.OK
    assert L.polylab_simplify_batched_workspace_bytes(1000, 9, 3, None) > L.polylab_simplify_workspace_bytes(1000, 3, None)
    assert L.polylab_matmul_simplify_workspace_bytes(1 << 30, 10, 10, 3, 3, 3, 3, None) == 0


def test_pow_simplify_host_side_checks(L):
    """polylab_pow_simplify: argument errors and the workspace query, no GPU involved."""
    from paper_2604_06575_b200 import binding as B
    cnt = ctypes.c_int64(-7)
    one = ctypes.c_void_p(16)
    f = L.polylab_pow_simplify
    p = B._Poly(16, 16, 10, 3)

    def call(poly=p, power=3, tol=0.0, opts=None, cap=100, cntp=ctypes.addressof(cnt), ws=one, wsb=1 << 30):
        return f(ctypes.byref(poly) if poly is not None else None, power, tol, opts, one, one, cap, cntp, ws, wsb, None)

    assert call(power=-1) == B.ERR_INVALID_ARGUMENT
    assert call(poly=None) == B.ERR_INVALID_ARGUMENT
    assert call(tol=float("nan")) == B.ERR_INVALID_ARGUMENT
    assert call(cntp=None) == B.ERR_INVALID_ARGUMENT
    assert call(poly=B._Poly(16, 16, 10, 0)) == B.ERR_INVALID_ARGUMENT
    assert call(ws=None) == B.ERR_INVALID_ARGUMENT
    assert call(wsb=1024) == B.ERR_WORKSPACE_TOO_SMALL
    o = B._Opts()
    o.term_stride, o.var_stride = 1, 10                      # strided operands are not supported by the power routine
    assert call(opts=ctypes.byref(o)) == B.ERR_INVALID_ARGUMENT
    o = B._Opts()
    bounds = (ctypes.c_uint32 * 3)(1, 1, 1)
    o.max_exp_host = ctypes.cast(bounds, ctypes.POINTER(ctypes.c_uint32))
    assert call(opts=ctypes.byref(o)) == B.ERR_INVALID_ARGUMENT
    assert call(poly=B._Poly(16, 16, 1 << 20, 3), cap=1 << 20) == B.ERR_INVALID_ARGUMENT     # a product could reach 2^30 terms
    q = L.polylab_pow_simplify_workspace_bytes
    assert q(200, 20, 1, 1000, None) == L.polylab_simplify_workspace_bytes(200, 20, None)
    assert q(200, 20, 3, 300_000, None) >= L.polylab_mul_simplify_workspace_bytes(300_000, 200, 20, None)
    assert q(200, 20, -1, 1000, None) == 0 and q(1 << 20, 3, 2, 1 << 20, None) == 0


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_2604_06575_b200 import binding as B
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(B.PolylabError, match="no CPU fallback"):
        B.lib()


def test_product_path_does_not_import_oracle():
    """The oracle is test infrastructure: nothing in the package may import or read it."""
    pkg = os.path.join(ROOT, "paper_2604_06575_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), fn
                assert "polylab_oracle" not in text, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2604_06575_b200", text, flags=re.M), fn

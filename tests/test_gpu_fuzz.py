"""-m gpu: a seeded fuzzer over every path of the library against the CPU oracle -- random variable counts (1..40), exponent
dtypes and ranges (keys of 0..256 bits), sizes around every threshold (one-block cap, tile sizes, table minimum), duplication
1..1000x, cancelling halves, coefficients spanning 40 decades, three tolerances; each input through the default path and
with the table, one-block, bucket, fused-pack and ranking choices forced on or off; products and batched calls on the same
draws.  (compute-sanitizer is not available on the GPU pool; this found the window-boundary bug of the cross-tile fix-up.)"""
import numpy as np
import pytest
import torch

from oracle import oracle, parity
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import dev

pytestmark = pytest.mark.gpu

FLAGSETS = [0, B.FLAG_NO_TABLE, B.FLAG_NO_SMALL, B.FLAG_NO_TABLE | B.FLAG_NO_SMALL, B.FLAG_DEBUG_FORCE_TABLE,
            B.FLAG_DEBUG_FORCE_TABLE | B.FLAG_DEBUG_FORCE_HASH, B.FLAG_DEBUG_FORCE_BUCKET, B.FLAG_SAFE_RANK,
            B.FLAG_NO_BUCKET | B.FLAG_NO_TABLE, B.FLAG_NO_FUSED_PACK]


def ok(res, c, e, what):
    rep = parity.check(res, c.cpu().numpy(), e.cpu().numpy())
    assert rep.ok, f"{what}: {rep}"


@pytest.mark.parametrize("seed", range(120))
def test_fuzz_all_paths(seed):
    r = np.random.default_rng(900_000 + seed)
    dtype = [np.uint8, np.uint16, np.uint32][int(r.integers(0, 3))]
    nvars = int(r.choice([1, 2, 3, 5, 8, 12, 17, 33, 40]))
    cap = {np.uint8: 256, np.uint16: 65536, np.uint32: 2 ** 32}[dtype]
    his = [int(min(cap, r.choice([1, 2, 3, 4, 16, 200, 256, 1000, 70000, 2 ** 31]))) for _ in range(nvars)]
    while sum(int(h - 1).bit_length() for h in his) > 256:
        his[int(r.integers(0, nvars))] = 2
    n = int(r.choice([1, 2, 33, 700, 4096, 4097, 8192, 8193, 20000, 40000, 90001, 300000]))
    dup = int(r.choice([1, 2, 4, 5, 50, 1000]))
    pool = np.stack([r.integers(0, h, size=max(1, n // dup)) for h in his], axis=1).astype(dtype)
    exps = np.ascontiguousarray(pool[r.integers(0, len(pool), size=n)])
    coef = r.standard_normal(n) * 10.0 ** r.integers(-20, 20, size=n) if seed % 5 == 0 else r.standard_normal(n)
    if seed % 4 == 0:                                               # p - p: every monomial cancels exactly
        coef[: n // 2] = -coef[n - n // 2:][::-1]
        exps[: n // 2] = exps[n - n // 2:][::-1]
    tol = [0.0, 1e-14, 0.5][seed % 3]
    res = oracle.simplify(coef, exps, tol)
    for fl in FLAGSETS:
        c, e = B.simplify(dev(coef), dev(exps), tol, flags=fl)
        ok(res, c, e, f"simplify flags {fl:#x} n {n} his {his}")
    # products of two draws with the same ranges (sums must fit the dtype)
    na, nb = int(r.choice([1, 7, 90, 200, 1100])), int(r.choice([1, 5, 64, 300]))
    hi2 = [max(1, min(h, cap // 2)) for h in his]
    if sum(int(2 * h - 2).bit_length() for h in hi2) <= 256:
        a = W.Poly(r.standard_normal(na), np.stack([r.integers(0, h, size=na) for h in hi2], axis=1).astype(dtype))
        b = W.Poly(r.standard_normal(nb), np.stack([r.integers(0, h, size=nb) for h in hi2], axis=1).astype(dtype))
        resm = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol)
        for fl in FLAGSETS:
            c, e = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, flags=fl)
            ok(resm, c, e, f"mul flags {fl:#x} {na}x{nb} his {hi2}")
    # the simplify input cut into random entries of a batch
    if n >= 2 and sum(int(h - 1).bit_length() for h in his) <= 250:
        ne = int(r.integers(1, 12))
        off = np.concatenate([[0], np.sort(r.integers(0, n + 1, size=ne - 1)), [n]]).astype(np.int64)
        gc, ge, go = B.simplify_batched(dev(coef), dev(exps), off, tol)
        for k in range(ne):
            rk = oracle.simplify(coef[off[k]:off[k + 1]], exps[off[k]:off[k + 1]], tol)
            ok(rk, gc[go[k]:go[k + 1]], ge[go[k]:go[k + 1]], f"batched entry {k} of {ne}")

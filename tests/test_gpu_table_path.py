"""-m gpu: the table path of the CUDA library (csrc/table.cu: like terms merged in a dense or hash table
with order-independent fixed-point accumulators, only the distinct monomials sorted) against the CPU oracle under the same
parity rule -- the paper's regime of heavy duplication (simplify(p_4^3): 2,000,376 raw terms -> 6188, PAPER.md:543, 584,
586) and BASELINE.json's configs 1-4 -- its abandonment when the input does not collapse, and the properties the
fixed-point sums add: bit-identical results under any permutation of the input and exact cancellation."""
import math

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import assert_parity, dev

pytestmark = pytest.mark.gpu

FT = B.FLAG_DEBUG_FORCE_TABLE
FH = B.FLAG_DEBUG_FORCE_TABLE | B.FLAG_DEBUG_FORCE_HASH


def run(p, tol, flags=0, **kw):
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, flags=flags, **kw)
    torch.cuda.synchronize()
    return c.cpu().numpy(), e.cpu().numpy(), st


def run_mul(a, b, tol, flags=0, **kw):
    c, e, st = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, return_stats=True, flags=flags, **kw)
    torch.cuda.synchronize()
    return c.cpu().numpy(), e.cpu().numpy(), st


def test_config1_dense_table():
    p, tol = W.config1()
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = run(p, tol)
    assert st.table_path == 1 and st.sort_passes == 0 and st.distinct == 256 and st.survivors == 256
    rep = assert_parity(res, c, e)
    assert rep.matched == 256
    c2, e2, st2 = run(p, tol, flags=FH)                        # the same through the hash table + a sort of 256 keys
    assert st2.table_path == 2 and st2.distinct == 256
    assert (e2 == e).all() and (c2.view(np.uint64) == c.view(np.uint64)).all()    # the sums do not depend on the table


def test_config2_dense_table_products():
    a, b, tol = W.config2()
    res = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol)
    c, e, st = run_mul(a, b, tol)
    assert st.table_path == 1 and st.key_bits == 18 and st.sort_terms == 4_000_000
    rep = assert_parity(res, c, e)
    assert rep.matched == int(res.keep.sum()) == len(c) and st.distinct == len(res.sum)
    c0, e0, st0 = run_mul(a, b, tol, flags=B.FLAG_NO_TABLE)
    assert st0.table_path == 0 and (e0 == e).all()


@pytest.mark.parametrize("n", [100_000, 1_000_003])
def test_config3_hash_table(n):
    p, tol = W.config3(n)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = run(p, tol)
    assert st.table_path == 2 and st.key_bits == 30 and st.distinct == len(res.sum) <= 7680 and st.table_fallback == 0
    assert_parity(res, c, e)


def test_config4_variant_b_hash_table_products():
    p, tol = W.config4()
    rc, re_ = B.expand(dev(p.coef), dev(p.exps), dev(p.coef), dev(p.exps))
    c, e, st = B.mul_simplify(rc, re_, dev(p.coef), dev(p.exps), tol, return_stats=True)
    assert st.table_path == 2 and st.sort_terms == 8_000_000
    c0, e0 = oracle.expand(p.coef, p.exps, p.coef, p.exps)
    res = oracle.mul_simplify(c0, e0, p.coef, p.exps.astype(e0.dtype), tol)
    assert_parity(res, c.cpu().numpy(), e.cpu().numpy())


@pytest.mark.parametrize("d", [2, 3, 4])
def test_paper_pd_cubed_one_shot(d):
    """The paper's Fig. 2 workload: simplify(p_d^3), 5 variables; raw p*p times p in one call.
    Closed form: C(5+3d, 5) terms, integer coefficients that sum to C(5+d, d)^3 -- bit-exact on the table path."""
    p = W.p_d(d)
    rc, re_ = B.expand(dev(p.coef), dev(p.exps), dev(p.coef), dev(p.exps))
    flags = 0 if p.nterms ** 3 >= 32768 else FT
    c, e, st = B.mul_simplify(rc, re_, dev(p.coef), dev(p.exps), 0.0, return_stats=True, flags=flags)
    c, e = c.cpu().numpy(), e.cpu().numpy()
    assert st.table_path == (2 if d == 3 else 1)               # d = 3: 2^20 slots for 175,616 products is not worth a dense table
    assert len(c) == math.comb(5 + 3 * d, 5) and c.sum() == float(p.nterms ** 3)
    assert (c == np.round(c)).all() and c.min() >= 1.0
    q = oracle.mul_simplify(p.coef, p.exps, p.coef, p.exps, 0.0)
    res = oracle.mul_simplify(*q.pruned, p.coef, p.exps.astype(np.uint32), 0.0)
    assert (e == res.pruned[1]).all() and (c == res.pruned[0]).all()


def test_not_collapsing_input_abandons_the_table():
    """Mostly distinct 60-bit keys: more than N/4 distinct monomials -> the insert pass raises `overflow`, the call goes on
    on the sort path with the keys it already packed."""
    r = np.random.default_rng(3)
    n = 400_000
    exps = r.integers(0, 1 << 15, size=(n, 4)).astype(np.uint16)
    exps[n // 2:] = exps[: n - n // 2]                          # every key twice: U = N/2
    p = W.Poly(r.standard_normal(n), exps)
    res = oracle.simplify(p.coef, p.exps, 0.0)
    c, e, st = run(p, 0.0)
    assert st.table_path == 0 and st.table_fallback == 1 and st.key_bits == 60
    assert_parity(res, c, e)
    # a collapse of exactly 4x is kept
    exps4 = np.concatenate([exps[: n // 4]] * 4)
    p4 = W.Poly(p.coef, np.ascontiguousarray(exps4))
    c, e, st = run(p4, 0.0)
    assert st.table_path == 2 and st.table_fallback == 0
    assert_parity(oracle.simplify(p4.coef, p4.exps, 0.0), c, e)


def test_permutation_invariance_is_bit_exact():
    """Integer accumulators: the sum does not depend on the order of the atomics, hence not on the order of the input."""
    p, tol = W.config3(500_000)
    c1, e1, st = run(p, tol)
    assert st.table_path == 2
    perm = np.random.default_rng(8).permutation(p.nterms)
    c2, e2, _ = run(W.Poly(p.coef[perm], np.ascontiguousarray(p.exps[perm])), tol)
    assert (e1 == e2).all() and (c1.view(np.uint64) == c2.view(np.uint64)).all()
    c3, e3, _ = run(p, tol)
    assert (c1.view(np.uint64) == c3.view(np.uint64)).all()
    # within 2 ulp of the correctly rounded sum (math.fsum) for every monomial: far inside 1e-12 * A_m
    res = oracle.simplify(p.coef, p.exps, tol)
    ulp = np.spacing(np.abs(res.sum))
    assert (np.abs(c1 - res.sum) <= 4 * ulp).all()
    # scaling by a power of two scales the result exactly
    c4, _, _ = run(W.Poly(p.coef * 2.0 ** -300, p.exps), 0.0)
    assert (c4 == c1 * 2.0 ** -300).all()


@pytest.mark.parametrize("flags", [FT, FH])
def test_exact_cancellation_and_dynamic_range(flags):
    """1e16 + 1 - 1e16 = 1 exactly (a plain fp64 sum in this order gives 0 or 2); a monomial whose terms span 600 binades;
    denormals; -0.0; zero coefficients; terms below tol that merge into a big sum (reading A4)."""
    exps = np.array([[1, 0], [1, 0], [1, 0],          # 1e16, 1, -1e16
                     [0, 2], [0, 2],                  # 1e300 + 1e-300
                     [3, 3], [3, 3],                  # denormals
                     [4, 0], [4, 0],                  # -0.0 + 0.0
                     [5, 5], [5, 5], [5, 5],          # p - p
                     [6, 1], [6, 1]], np.uint8)       # 1e-20 merges into 1.0
    coef = np.array([1e16, 1.0, -1e16, 1e300, 1e-300, 5e-324, 1.5e-323, -0.0, 0.0, 0.7, -0.2, -0.5, 1e-20, 1.0])
    c, e, st = run(W.Poly(coef, exps), 0.0, flags=flags)
    assert st.table_path == (1 if flags == FT else 2)
    got = {tuple(r): v for r, v in zip(e.tolist(), c.tolist())}
    assert got[(1, 0)] == 1.0
    assert got[(0, 2)] == 1e300
    assert got[(3, 3)] == 2e-323
    assert (4, 0) not in got
    assert got[(6, 1)] == 1.0                         # 1 + 1e-20 rounds to 1
    assert abs(got.get((5, 5), 0.0)) <= 1e-12 * 1.4   # 0.7 - 0.2 - 0.5: exactly 2^-54-ish or 0, inside the exemption band
    assert_parity(oracle.simplify(coef, exps, 0.0), c, e)
    # tolerance semantics on the table path (reading A2): |s| == tol dropped, the next double kept
    exps2 = np.array([[1], [2], [3], [3]], np.uint8)
    t = 0.75
    c, e, _ = run(W.Poly(np.array([0.75, np.nextafter(0.75, 1.0), 0.5, 0.25]), exps2), t, flags=flags)
    assert e.tolist() == [[2]] and c[0] == np.nextafter(0.75, 1.0)


@pytest.mark.parametrize("flags", [FT, FH])
def test_nonfinite_coefficients_on_the_table_path(flags):
    """Reading A12: non-finite values propagate through a monomial's sum as in a plain IEEE sum; NaN sums are dropped."""
    inf = float("inf")
    exps = np.array([[0], [0], [1], [1], [1], [2], [2], [2], [3], [3], [4]], np.uint8)
    coef = np.array([inf, 1.0, 2.0, -inf, 3.0, inf, -inf, 4.0, float("nan"), 7.0, 5.0])
    c, e, st = run(W.Poly(coef, exps), 0.0, flags=flags)
    assert e.tolist() == [[0], [1], [4]] and c.tolist() == [inf, -inf, 5.0]
    oc, oe = oracle.simplify(coef, exps, 0.0).pruned            # (the parity rule's |g - s| is not defined for infinities)
    assert oe.tolist() == e.tolist() and oc.tolist() == c.tolist()


@pytest.mark.parametrize("flags", [FT, FH])
@pytest.mark.parametrize("n", [1, 33, 5000, 40_000])
def test_forced_table_small_and_all_equal(n, flags):
    r = np.random.default_rng(n)
    coef = r.standard_normal(n)
    exps = np.tile(np.array([[3, 1, 4, 1, 5]], np.uint8), (n, 1))
    c, e, st = run(W.Poly(coef, exps), 0.0, flags=flags)
    assert st.table_path in (1, 2) and len(c) == 1
    assert abs(c[0] - math.fsum(coef.tolist())) <= 4 * np.spacing(abs(c[0]))
    p, tol = W.config1(n)
    c, e, st = run(p, tol, flags=flags)
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


def test_table_path_capacity_strides_dtypes_and_bounds():
    p, tol = W.config3(200_000, dtype=np.uint32)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = run(p, tol)
    assert st.table_path == 2 and e.dtype == np.uint32
    assert_parity(res, c, e)
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p.coef), dev(p.exps), tol, out_capacity=100)
    assert ei.value.status == B.ERR_OUTPUT_TOO_SMALL
    # column-major exponents (MATLAB's pow, reading A13)
    cm = dev(np.ascontiguousarray(p.exps.T)).T
    c2, e2, st2 = B.simplify(dev(p.coef), cm, tol, return_stats=True)
    assert st2.table_path == 2 and (e2.cpu().numpy() == e).all() and (c2.cpu().numpy() == c).all()
    # caller bounds: loose ones still give the same polynomial; a violated one is reported
    c3, e3, st3 = B.simplify(dev(p.coef), dev(p.exps), tol, max_exp=[7] * 10, return_stats=True)
    assert st3.table_path == 2 and (e3.cpu().numpy() == e).all() and (c3.cpu().numpy() == c).all()
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p.coef), dev(p.exps), tol, max_exp=[3] * 10)
    assert ei.value.status == B.ERR_EXPONENT_RANGE
    # dense table with a capacity error
    p1, tol1 = W.config1()
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p1.coef), dev(p1.exps), tol1, out_capacity=10)
    assert ei.value.status == B.ERR_OUTPUT_TOO_SMALL


def test_hash_table_with_many_distinct_keys():
    """2^20 - ish distinct monomials of 40 bits among 8e6 terms: the accumulators beyond the first 8192 ordinals live in
    global memory (red.global.add.u64)."""
    r = np.random.default_rng(12)
    n, u = 8_000_000, 900_000
    pool = r.integers(0, 256, size=(u, 5), dtype=np.uint8)
    exps = np.ascontiguousarray(pool[r.integers(0, u, size=n)])
    p = W.Poly(r.standard_normal(n), exps)
    res = oracle.simplify(p.coef, p.exps, 0.0)
    c, e, st = run(p, 0.0)
    assert st.table_path == 2 and st.distinct == len(res.sum)
    assert_parity(res, c, e)

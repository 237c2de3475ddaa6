"""More pins of the oracle: brute force through a dense array, exact sums, invariants,
tolerance semantics.  Expected values never come from the oracle itself or the CUDA path."""
import itertools
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle
from paper_2604_06575_b200 import workloads as W

METHODS = ["hash", "sortscan"]


def _dense_brute_force(coef, exps, shape):
    """No hashing, no sorting, no keys: accumulate into a dense array indexed by the exponent tuple
    (exact Fractions), read out in nested-loop order = ascending lex with variable 0 outermost."""
    dense = np.empty(shape, dtype=object)
    hit = np.zeros(shape, dtype=bool)
    for idx in itertools.product(*[range(s) for s in shape]):
        dense[idx] = Fraction(0)
    for c, row in zip(coef, exps.tolist()):
        dense[tuple(row)] += Fraction(float(c))
        hit[tuple(row)] = True
    out = []
    for idx in itertools.product(*[range(s) for s in shape]):
        if hit[idx]:
            out.append((idx, dense[idx]))
    return out


@pytest.mark.parametrize("method", METHODS)
def test_exhaustive_tiny_multisets(method):
    """All multisets of <= 4 terms from a 2x2 exponent grid with coefficients in {-1,0,1,0.5}."""
    grid = list(itertools.product(range(2), repeat=2))
    coefs = [-1.0, 0.0, 1.0, 0.5]
    atoms = [(g, c) for g in grid for c in coefs]
    n_cases = 0
    for k in range(0, 5):
        for combo in itertools.combinations_with_replacement(range(len(atoms)), k):
            rows = np.array([atoms[i][0] for i in combo], np.uint8).reshape(k, 2)
            c = np.array([atoms[i][1] for i in combo], float)
            res = oracle.simplify(c, rows, 0.0, method=method)
            want = _dense_brute_force(c, rows, (2, 2))
            assert [tuple(r) for r in res.rows.tolist()] == [w[0] for w in want]
            assert res.sum.tolist() == [float(w[1]) for w in want]
            assert res.keep.tolist() == [w[1] != 0 for w in want]
            n_cases += 1
    assert n_cases == sum(math.comb(16 + k - 1, k) for k in range(5))


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("nvars,emax,n", [(1, 7, 200), (2, 3, 500), (3, 3, 2000)])
def test_dense_brute_force_random(method, nvars, emax, n):
    r = np.random.default_rng(7 + nvars)
    exps = r.integers(0, emax + 1, size=(n, nvars)).astype(np.uint16)
    coef = r.integers(-8, 9, size=n) / 4.0           # dyadic: every sum is exact in fp64
    res = oracle.simplify(coef, exps, 0.0, method=method)
    want = _dense_brute_force(coef, exps, (emax + 1,) * nvars)
    assert [tuple(x) for x in res.rows.tolist()] == [w[0] for w in want]
    assert res.sum.tolist() == [float(w[1]) for w in want]
    assert res.abs.tolist() == [float(sum(abs(Fraction(float(c))) for c, row in zip(coef, exps.tolist())
                                          if tuple(row) == w[0])) for w in want]
    assert res.count.sum() == n


def _dict_fsum(coef, exps):
    groups = {}
    for c, row in zip(coef.tolist(), exps.tolist()):
        groups.setdefault(tuple(row), []).append(c)
    keys = sorted(groups)
    return keys, [math.fsum(groups[k]) for k in keys], [math.fsum(abs(x) for x in groups[k]) for k in keys]


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("cfg", ["c1", "c3", "c5"])
def test_sums_against_fsum(method, cfg):
    """s_m within 1 ulp of the correctly rounded exact sum (math.fsum); order = Python tuple order."""
    if cfg == "c1":
        p, tol = W.config1(20_000)
    elif cfg == "c3":
        p, tol = W.config3(30_000)
    else:
        p, tol = W.config5(20_000)
    res = oracle.simplify(p.coef, p.exps, tol, method=method)
    keys, sums, abss = _dict_fsum(p.coef, p.exps)
    assert [tuple(r) for r in res.rows.tolist()] == keys
    for got, want, a in zip(res.sum.tolist(), sums, abss):
        assert abs(got - want) <= math.ulp(want) + 4 * 2.0 ** -53 * 2.0 ** -53 * a, (got, want)
    np.testing.assert_allclose(res.abs, abss, rtol=1e-13)


def test_ill_conditioned_sum_is_compensated():
    """1e16 + 1 - 1e16 + ... : naive left-to-right summation loses the ones, the oracle does not."""
    coef = np.array([1e16, 1.0, -1e16, 1.0, 1e-3, 1e16, -1e16])
    exps = np.zeros((7, 2), np.uint8)
    for method in METHODS:
        res = oracle.simplify(coef, exps)
        assert res.sum[0] == math.fsum(coef.tolist()) == 2.001


def test_product_against_fractions():
    """mul_simplify on dyadic coefficients equals exact rational polynomial multiplication."""
    r = np.random.default_rng(11)
    a = (r.integers(-16, 17, 40) / 8.0, r.integers(0, 3, (40, 3)).astype(np.uint8))
    b = (r.integers(-16, 17, 30) / 8.0, r.integers(0, 4, (30, 3)).astype(np.uint8))
    exact = {}
    for ca, ra in zip(a[0].tolist(), a[1].tolist()):
        for cb, rb in zip(b[0].tolist(), b[1].tolist()):
            k = tuple(x + y for x, y in zip(ra, rb))
            exact[k] = exact.get(k, Fraction(0)) + Fraction(ca) * Fraction(cb)
    res = oracle.mul_simplify(a[0], a[1], b[0], b[1])
    assert [tuple(x) for x in res.rows.tolist()] == sorted(exact)
    assert res.sum.tolist() == [float(exact[k]) for k in sorted(exact)]
    assert res.keep.tolist() == [exact[k] != 0 for k in sorted(exact)]
    assert int(res.count.sum()) == 40 * 30


def test_expand_layout_and_single_rounding():
    """Term (i,j) at i*nb+j; coefficient = one IEEE multiplication; row = a_i + b_j."""
    r = np.random.default_rng(3)
    ca, cb = r.standard_normal(7), r.standard_normal(5)
    ea, eb = r.integers(0, 200, (7, 4)).astype(np.uint8), r.integers(0, 200, (5, 4)).astype(np.uint8)
    pc, pr = oracle.expand(ca, ea, cb, eb)
    assert pc.tolist() == [x * y for x in ca.tolist() for y in cb.tolist()]
    assert pr.tolist() == [[p + q for p, q in zip(x, y)] for x in ea.tolist() for y in eb.tolist()]  # sums > 255 kept


@pytest.mark.parametrize("method", METHODS)
def test_p_minus_p_is_zero(method):
    p, _ = W.config1(5000)
    coef = np.concatenate([p.coef, -p.coef])
    exps = np.concatenate([p.exps, p.exps])
    perm = np.random.default_rng(0).permutation(len(coef))
    res = oracle.simplify(coef[perm], exps[perm], 0.0, method=method)
    assert res.keep.sum() == 0 and np.all(res.sum == 0.0)
    assert len(res.pruned[0]) == 0


def test_evaluation_invariance_and_product_rule():
    a, b, _ = W.config2(60)
    res = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps)
    c, rows = res.pruned
    for x in W.eval_points(6, 8):
        va, _ = oracle.evaluate(a.coef, a.exps, x)
        vb, _ = oracle.evaluate(b.coef, b.exps, x)
        vr, ar = oracle.evaluate(c, rows, x)
        assert abs(vr - va * vb) <= 1e-12 * ar + 1e-300
    # commutativity: identical sets, sums equal up to rounding of the summation order
    res2 = oracle.mul_simplify(b.coef, b.exps, a.coef, a.exps)
    assert res.rows.tolist() == res2.rows.tolist()
    assert np.all(np.abs(res.sum - res2.sum) <= 1e-15 * res.abs)
    # simplify leaves p(x) unchanged
    p, _ = W.config3(4000)
    sc, sr = oracle.simplify(p.coef, p.exps).pruned
    for x in W.eval_points(10, 4):
        v0, a0 = oracle.evaluate(p.coef, p.exps, x)
        v1, _ = oracle.evaluate(sc, sr, x)
        assert abs(v0 - v1) <= 1e-12 * a0


@pytest.mark.parametrize("method", METHODS)
def test_idempotence_permutation_scaling(method):
    p, _ = W.config4()
    res = oracle.simplify(p.coef, p.exps, 0.0, method=method)
    c, r = res.pruned
    again = oracle.simplify(c, r, 0.0, method=method)
    assert again.rows.tolist() == r.tolist() and again.sum.tolist() == c.tolist()
    assert [tuple(x) for x in r.tolist()] == sorted({tuple(x) for x in p.exps.tolist()})
    perm = np.random.default_rng(5).permutation(p.nterms)
    res_p = oracle.simplify(p.coef[perm], p.exps[perm], 0.0, method=method)
    assert res_p.rows.tolist() == res.rows.tolist()
    assert np.all(np.abs(res_p.sum - res.sum) <= 2.0 ** -52 * res.abs)
    res_s = oracle.simplify(p.coef * 2.0 ** 40, p.exps, 0.0, method=method)
    assert (res_s.sum == res.sum * 2.0 ** 40).all()
    # strictly ascending, sum of coefficients = p(1,...,1)
    assert abs(res.sum.sum() - math.fsum(p.coef.tolist())) <= 1e-13 * np.abs(p.coef).sum()


@pytest.mark.parametrize("method", METHODS)
def test_tolerance_semantics(method):
    """Reading A2: keep iff |s| > tol (absolute, strict); A4: prune after merging only; A12: NaN dropped."""
    tol = 0.25
    up = math.nextafter(tol, 1.0)
    coef = np.array([0.25, -0.25, up, -up, 0.125, 0.125, 0.1, 100.0, 1.0, -1.0, float("nan")])
    exps = np.array([[0], [1], [2], [3], [4], [4], [5], [5], [6], [6], [7]], np.uint8)
    res = oracle.simplify(coef, exps, tol, method=method)
    assert res.rows[:, 0].tolist() == list(range(8))
    #                     =tol   =-tol  tol+ulp -(tol+ulp) 2*.125=tol small+big  cancel  NaN
    assert res.keep.tolist() == [False, False, True, True, False, True, False, False]
    assert res.sum[5] == 100.1
    # tol = 0: exact zeros and -0.0 are dropped, everything else kept
    res0 = oracle.simplify(np.array([-0.0, 5e-324, 1.0, -1.0]), np.array([[0], [1], [2], [2]], np.uint8), 0.0, method=method)
    assert res0.keep.tolist() == [False, True, False]


@pytest.mark.parametrize("method", METHODS)
def test_nonfinite_coefficients_propagate(method):
    """Reading A12: +-inf propagates through a monomial's sum like in a plain sum (kept: |inf| > tol);
    inf + (-inf) = NaN and NaN fail the predicate and are dropped.  The values are those of IEEE addition."""
    inf = float("inf")
    coef = np.array([inf, 1.0, 2.0, -inf, 3.0, inf, -inf, 4.0, 1.5, float("nan"), 7.0])
    exps = np.array([[0], [0], [1], [1], [1], [2], [2], [2], [3], [4], [4]], np.uint8)
    res = oracle.simplify(coef, exps, 0.5, method=method)
    assert res.rows[:, 0].tolist() == [0, 1, 2, 3, 4]
    assert res.sum[0] == inf and res.sum[1] == -inf and math.isnan(res.sum[2]) and res.sum[3] == 1.5 and math.isnan(res.sum[4])
    assert res.keep.tolist() == [True, True, False, True, False]
    assert res.abs[0] == inf and res.count.tolist() == [2, 3, 3, 1, 2]


@pytest.mark.parametrize("method", METHODS)
def test_exponent_dtypes_and_empty(method):
    r = np.random.default_rng(2)
    rows = r.integers(0, 200, (300, 5))
    coef = r.standard_normal(300)
    ref = oracle.simplify(coef, rows.astype(np.uint32), method=method)
    for dt in (np.uint8, np.uint16, np.int64):
        got = oracle.simplify(coef, rows.astype(dt), method=method)
        assert got.rows.tolist() == ref.rows.tolist() and got.sum.tolist() == ref.sum.tolist()
    big = oracle.simplify([1.0, 2.0, 3.0], np.array([[70000, 0], [256, 1], [70000, 0]], np.uint32), method=method)
    assert big.rows.tolist() == [[256, 1], [70000, 0]] and big.sum.tolist() == [2.0, 4.0]
    empty = oracle.simplify(np.zeros(0), np.zeros((0, 3), np.uint8), method=method)
    assert empty.rows.shape == (0, 3) and len(empty.sum) == 0
    with pytest.raises(ValueError):
        oracle.simplify([1.0], np.array([[-1, 0]]))
    with pytest.raises(ValueError):
        oracle.simplify([1.0, 2.0], np.array([[1, 0]], np.uint8))

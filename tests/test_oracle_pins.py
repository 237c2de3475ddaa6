"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests compares the oracle with itself or with the CUDA path: the
expected values are the paper's worked examples (tests/golden/paper_examples.json,
each with its citation), closed forms (multinomial coefficients, C(n+k-1,k),
C(5+3d,5)), brute force through a dense array (no hashing, no sorting), exact
rational arithmetic and math.fsum.  SURVEY.md 8(c) "What pins each part".
"""
import itertools
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle
from paper_2604_06575_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_examples.json")
with open(GOLDEN) as f:
    PAPER = json.load(f)

METHODS = ["hash", "sortscan"]


def _as_set(coef, rows):
    return {tuple(int(e) for e in r): float(c) for c, r in zip(coef, rows)}


def _run_example(ex, method):
    if ex["op"] == "simplify":
        res = oracle.simplify(np.array(ex["coef"], float), np.array(ex["exps"], np.uint8), ex["tol"], method=method)
    else:
        # products: expand with the oracle, then merge with the method under test
        pc, pr = oracle.expand(np.array(ex["a_coef"], float), np.array(ex["a_exps"], np.uint8),
                               np.array(ex["b_coef"], float), np.array(ex["b_exps"], np.uint8))
        res = oracle.simplify(pc, pr, ex["tol"], method=method)
    return res.pruned


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("ex", PAPER["examples"], ids=[e["name"] for e in PAPER["examples"]])
def test_paper_worked_examples(ex, method):
    coef, rows = _run_example(ex, method)
    want_c, want_r = ex["out_coef"], ex["out_exps"]
    if ex["ordered"]:
        # machine-printed transcript: order is part of the pin (reading A1)
        assert rows.tolist() == want_r, ex["cite"]
        assert coef.tolist() == [float(c) for c in want_c], ex["cite"]
    else:
        assert _as_set(coef, rows) == _as_set(want_c, want_r), ex["cite"]


@pytest.mark.parametrize("ex", [e for e in PAPER["examples"] if e["op"] == "mul_simplify"],
                         ids=lambda e: e["name"])
def test_paper_products_via_mul_simplify(ex):
    res = oracle.mul_simplify(np.array(ex["a_coef"], float), np.array(ex["a_exps"], np.uint8),
                              np.array(ex["b_coef"], float), np.array(ex["b_exps"], np.uint8), ex["tol"])
    coef, rows = res.pruned
    assert _as_set(coef, rows) == _as_set(ex["out_coef"], ex["out_exps"]), ex["cite"]


def test_paper_subs_example_full():
    """us = 3(z1+1)^2 + 5 z2 = 3 + 6 z1 + 3 z1^2 + 5 z2."""
    sq = oracle.mul_simplify([1, 1], np.array([[1, 0], [0, 0]], np.uint8), [1, 1], np.array([[1, 0], [0, 0]], np.uint8))
    c, r = sq.pruned
    coef = np.concatenate([3.0 * c, [5.0]])
    rows = np.concatenate([r, np.array([[0, 1]], np.uint32)])
    oc, orow = oracle.simplify(coef, rows).pruned
    assert _as_set(oc, orow) == {(0, 0): 3.0, (1, 0): 6.0, (2, 0): 3.0, (0, 1): 5.0}


@pytest.mark.parametrize("ex", PAPER["eval"], ids=lambda e: e["name"])
def test_paper_eval(ex):
    v, a = oracle.evaluate(np.array(ex["coef"], float), np.array(ex["exps"], np.uint8), ex["x"])
    assert v == ex["value"], ex["cite"]
    assert a == sum(abs(c) * math.prod(x ** e for x, e in zip(ex["x"], row)) for c, row in zip(ex["coef"], ex["exps"]))


def test_paper_grad_norm_quartic():
    """f = x1^4+2x1^2x2^2+x2^4+x3^2+3x4+1 at x0=(0.3,0.2,0.4,0.1): info.grad_norm = 3.110491e+00
    (PAPER.md:481-509).  The gradient's four components are polynomials typed in by hand here and
    evaluated by the oracle's evaluator: pins oracle_eval on non-integer points."""
    x0 = [0.3, 0.2, 0.4, 0.1]
    comps = [
        ([4, 4], [[3, 0, 0, 0], [1, 2, 0, 0]]),
        ([4, 4], [[2, 1, 0, 0], [0, 3, 0, 0]]),
        ([2], [[0, 0, 1, 0]]),
        ([3], [[0, 0, 0, 0]]),
    ]
    g = [oracle.evaluate(np.array(c, float), np.array(e, np.uint8), x0)[0] for c, e in comps]
    assert f"{math.sqrt(sum(v * v for v in g)):.6e}" == "3.110491e+00"


@pytest.mark.parametrize("ex", PAPER["counts"], ids=lambda e: e["name"])
def test_monolist_counts(ex):
    rows = W.monolist(ex["nvars"], ex["degree"])
    assert rows.shape[0] == ex["count"] == math.comb(ex["nvars"] + ex["degree"], ex["degree"]), ex["cite"]
    assert len({tuple(r) for r in rows.tolist()}) == ex["count"]
    assert int(rows.sum(axis=1).max()) == ex["degree"]


# ---------------------------------------------------------------- closed form 1: multinomials

def _power(coef, exps, k, method="hash"):
    """p^k by chained products, merged after each multiplication."""
    c, r = np.asarray(coef, float), np.asarray(exps, np.uint32)
    bc, br = c, r
    for _ in range(k - 1):
        pc, pr = oracle.expand(c, r.astype(np.uint32), bc, br)
        c, r = oracle.simplify(pc, pr, 0.0, method=method).pruned
    return c, r


@pytest.mark.parametrize("n,k", [(2, 2), (2, 6), (3, 3), (3, 5), (5, 4), (8, 3), (8, 4)])
def test_multinomial_closed_form(n, k):
    """(x1+...+xn)^k has C(n+k-1,k) terms; coefficient of x^alpha is k!/(alpha_1!...alpha_n!).
    All integers < 2^53, so exact in any summation order (north_star; SURVEY 8(c) closed form 1)."""
    c, r = _power(np.ones(n), np.eye(n, dtype=np.uint32), k)
    assert len(c) == math.comb(n + k - 1, k)
    for coef, row in zip(c, r.tolist()):
        assert sum(row) == k
        want = math.factorial(k)
        for e in row:
            want //= math.factorial(e)
        assert coef == float(want), (row, coef, want)
    assert r.tolist() == sorted(r.tolist())          # ascending lexicographic, variable 0 first
    assert c.sum() == float(n ** k)


@pytest.mark.parametrize("n,k", [(3, 4), (4, 5)])
def test_multinomial_one_shot_equals_chained(n, k):
    """Expanding all n^k raw terms at once and merging gives the same integers."""
    tuples = np.array(list(itertools.product(range(n), repeat=k)))
    rows = np.zeros((len(tuples), n), np.uint8)
    for j in range(k):
        np.add.at(rows, (np.arange(len(tuples)), tuples[:, j]), 1)
    for method in METHODS:
        c, r = oracle.simplify(np.ones(len(tuples)), rows, 0.0, method=method).pruned
        c2, r2 = _power(np.ones(n), np.eye(n, dtype=np.uint32), k)
        assert r.tolist() == r2.tolist() and c.tolist() == c2.tolist()


# ---------------------------------------------------------------- closed form 2: the paper's p_d^3

@pytest.mark.parametrize("d,nterms,csum", [(2, 462, 9261), (3, 2002, 175616)])
def test_paper_pd_cubed(d, nterms, csum):
    """p_d = sum_{|a|<=d} x^a in 5 variables: p_d^3 has C(5+3d,5) terms, integer
    coefficients summing to C(5+d,d)^3; for |alpha| <= d the coefficient is prod_v C(alpha_v+2, 2)."""
    p = W.p_d(d)
    assert p.nterms == math.comb(5 + d, d)
    c, r = _power(p.coef, p.exps, 3)
    assert len(c) == nterms == math.comb(5 + 3 * d, 5)
    assert c.sum() == float(csum) == float(p.nterms ** 3)
    as_map = _as_set(c, r)
    assert as_map[(0, 0, 0, 0, 0)] == 1.0
    for v in range(5):
        top = [0] * 5
        top[v] = 3 * d
        assert as_map[tuple(top)] == 1.0
    for row, coef in as_map.items():
        assert coef == int(coef) and coef > 0
        if sum(row) <= d:
            assert coef == float(math.prod(math.comb(e + 2, 2) for e in row)), row
    # intermediate p_d^2 has C(5+2d,5) terms
    c2, _ = _power(p.coef, p.exps, 2)
    assert len(c2) == math.comb(5 + 2 * d, 5)


def test_paper_pd_cubed_brute_force_triples():
    """Every coefficient of p_2^3 equals the number of ordered triples (b1,b2,b3), |bi|<=2, summing
    to alpha -- counted here with plain Python dict arithmetic on tuples."""
    d = 2
    base = [tuple(r) for r in W.monolist(5, d).tolist()]
    counts = {}
    for b1 in base:
        for b2 in base:
            s12 = tuple(x + y for x, y in zip(b1, b2))
            for b3 in base:
                a = tuple(x + y for x, y in zip(s12, b3))
                counts[a] = counts.get(a, 0) + 1
    p = W.p_d(d)
    c, r = _power(p.coef, p.exps, 3)
    assert _as_set(c, r) == {k: float(v) for k, v in counts.items()}
    # one-shot: all 21^3 raw terms at once
    pc, pr = oracle.expand(p.coef, p.exps, p.coef, p.exps)
    pc, pr = oracle.expand(pc, pr, p.coef, p.exps.astype(np.uint32))
    assert len(pc) == 9261
    for method in METHODS:
        c1, r1 = oracle.simplify(pc, pr, 0.0, method=method).pruned
        assert r1.tolist() == r.tolist() and c1.tolist() == c.tolist()

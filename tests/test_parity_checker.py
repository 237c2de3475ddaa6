"""The parity rule (north_star) as implemented by oracle/parity.py: each clause must
fire on a hand-made violation, and the workload generators must have the stated structure."""
import math

import numpy as np
import pytest

from oracle import oracle, parity
from paper_2604_06575_b200 import workloads as W


def _base():
    coef = np.array([1.0, 2.0, 3.0, -3.0, 0.5, 1e-20])
    exps = np.array([[0, 1], [0, 1], [1, 0], [1, 0], [2, 2], [3, 0]], np.uint8)
    return oracle.simplify(coef, exps, 1e-14)


def test_accepts_correct_and_band():
    res = _base()
    c, r = res.pruned
    assert r.tolist() == [[0, 1], [2, 2]]
    rep = parity.check(res, c, r)
    assert rep.ok and rep.matched == 2
    # (1,0) cancels exactly: |0 - tol| = 1e-14 > beta = 6e-12?  beta = 1e-12*6 -> exempt; may be present
    rep = parity.check(res, [3.0, 1e-15, 0.5], [[0, 1], [1, 0], [2, 2]])
    assert rep.ok and rep.exempt >= 1
    # coefficient perturbed inside / outside the bound 1e-12 * A_m (A = 3)
    assert parity.check(res, [3.0 + 2e-12, 0.5], r).ok
    assert not parity.check(res, [3.0 + 4e-12, 0.5], r).ok


def test_rejects_violations():
    res = _base()
    c, r = res.pruned
    assert not parity.check(res, c[::-1], r[::-1]).ok                       # order
    assert not parity.check(res, c[:1], r[:1]).ok                           # missing monomial
    assert not parity.check(res, [3.0, 0.5, 7.0], [[0, 1], [2, 2], [2, 3]]).ok   # invented monomial
    assert not parity.check(res, [3.0, 3.0, 0.5], [[0, 1], [0, 1], [2, 2]]).ok   # duplicate
    assert not parity.check(res, [3.0, 0.5, 1e-20], [[0, 1], [2, 2], [3, 0]]).ok  # should be pruned (A tiny)
    assert not parity.check(res, [float("nan"), 0.5], r).ok
    assert parity.check(res, c[:1], r[:1], subset_of_oracle=True).ok


def test_empty_cases():
    res = oracle.simplify(np.zeros(0), np.zeros((0, 2), np.uint8))
    assert parity.check(res, np.zeros(0), np.zeros((0, 2), np.uint8)).ok
    assert not parity.check(res, [1.0], [[0, 0]]).ok


# ------------------------------------------------------------------ workload generators

def test_config_shapes():
    p, tol = W.config1(10_000)
    assert p.exps.shape == (10_000, 4) and p.exps.max() == 3 and tol == 0.0 and np.abs(p.coef).max() <= 1
    assert len({tuple(r) for r in p.exps.tolist()}) == 256
    a, b, _ = W.config2(500)
    assert a.exps.shape == b.exps.shape == (500, 6) and a.exps.max() == 3
    p, _ = W.config3(20_000)
    assert ((p.exps > 0).sum(axis=1) == 3).all() and p.exps.max() == 4 and p.exps[p.exps > 0].min() == 1
    assert len({tuple(r) for r in p.exps.tolist()}) <= math.comb(10, 3) * 64      # reading A15: 7680
    p, _ = W.config3u(5000)
    assert p.exps.dtype == np.uint16 and ((p.exps > 0).sum(axis=1) == 3).all() and p.exps.max() > 255
    p, _ = W.config4()
    assert p.exps.shape == (200, 20) and p.exps.sum(axis=1).max() == 2 and p.exps.sum(axis=1).min() == 0
    p, tol = W.config5(40_000)
    assert tol == 1e-14 and p.exps.shape == (40_000, 16)
    res = oracle.simplify(p.coef, p.exps, tol)
    assert len(res.sum) == 4000 and (res.count == 10).all()           # pool of N/10, each exactly 10 times
    assert res.keep.sum() == 2000 and (res.sum[~res.keep] == 0.0).all()   # half cancels exactly (A18)


def test_generators_are_seeded():
    a1, _ = W.config3(1000)
    a2, _ = W.config3(1000)
    a3, _ = W.config3(1000, seed_offset=1)
    assert (a1.exps == a2.exps).all() and (a1.coef == a2.coef).all()
    assert not (a1.exps == a3.exps).all()

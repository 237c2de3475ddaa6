"""-m gpu: polylab_pow_simplify (the paper's mpower on a scalar polynomial, intermediates kept on the
device) against closed forms and against the oracle's chain of products."""
import math

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import assert_parity, dev

pytestmark = pytest.mark.gpu


def gpu_pow(p, k, tol=0.0, **kw):
    c, e = B.pow_simplify(dev(p.coef), dev(p.exps), k, tol, **kw)[:2]
    torch.cuda.synchronize()
    return c.cpu().numpy(), e.cpu().numpy()


def oracle_pow(p, k, tol=0.0):
    """Left-to-right chain, intermediates merged at tolerance 0, the last product pruned with tol (the ABI's definition)."""
    c, e = p.coef, p.exps
    for step in range(2, k + 1):
        res = oracle.mul_simplify(c, e, p.coef, p.exps, tol if step == k else 0.0)
        c, e = res.pruned
        e = e.astype(p.exps.dtype)
    return res


@pytest.mark.parametrize("n,k", [(2, 7), (3, 5), (5, 4), (8, 3)])
def test_multinomial_theorem(n, k):
    """(x1+...+xn)^k: C(n+k-1,k) terms with multinomial coefficients, bit-exact (north_star's closed form)."""
    base = W.Poly(np.ones(n), np.eye(n, dtype=np.uint8))
    c, e = gpu_pow(base, k)
    assert len(c) == math.comb(n + k - 1, k)
    assert e.tolist() == sorted(e.tolist())
    for coef, row in zip(c, e.tolist()):
        want = math.factorial(k)
        for x in row:
            want //= math.factorial(x)
        assert coef == float(want)


@pytest.mark.parametrize("d", [2, 3, 4])
def test_paper_pd_cubed(d):
    """simplify(p_d^3), 5 variables: C(5+3d,5) terms, integer coefficients summing to C(5+d,d)^3."""
    p = W.p_d(d)
    c, e = gpu_pow(p, 3)
    assert len(c) == math.comb(5 + 3 * d, 5)
    assert c.sum() == float(p.nterms ** 3) and (c == np.round(c)).all() and c.min() >= 1.0


def test_config4_cube_matches_the_oracle_chain():
    p, tol = W.config4()
    c, e = gpu_pow(p, 3, tol, out_capacity=300_000)
    assert_parity(oracle_pow(p, 3, tol), c, e)
    c2, e2 = gpu_pow(p, 2, tol)
    assert_parity(oracle.mul_simplify(p.coef, p.exps, p.coef, p.exps, tol), c2, e2)


def test_small_powers_errors_and_zero():
    p, _ = W.config4()
    c, e = gpu_pow(p, 0)
    assert c.tolist() == [1.0] and e.tolist() == [[0] * 20]
    c, e = gpu_pow(p, 1)
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)
    with pytest.raises(B.PolylabError) as ei:                       # the square alone has thousands of terms
        gpu_pow(p, 3, out_capacity=500)
    assert ei.value.status == B.ERR_OUTPUT_TOO_SMALL
    z = W.Poly(np.array([1.0, -1.0]), np.array([[1, 2], [1, 2]], np.uint8))     # p = 0 after merging
    c, e = gpu_pow(z, 4)
    assert len(c) == 0
    big = W.Poly(np.ones(1), np.array([[100]], np.uint8))           # x^100 cubed does not fit uint8
    with pytest.raises(B.PolylabError) as ei:
        gpu_pow(big, 3)
    assert ei.value.status == B.ERR_EXPONENT_RANGE
    c, e = gpu_pow(W.Poly(np.array([2.0]), np.array([[100]], np.uint16)), 3)
    assert c.tolist() == [8.0] and e.tolist() == [[300]]


@pytest.mark.parametrize("k", [4, 6, 8])
def test_higher_powers_match_the_oracle_chain(k):
    """The powers stay packed between the products (one key layout sized for degree k * max): k - 1 products, each against
    the oracle's chain; the last product's output is unpacked and pruned with tol."""
    r = np.random.default_rng(k)
    p = W.Poly(r.uniform(-1.0, 1.0, 12), r.integers(0, 3, size=(12, 4)).astype(np.uint8))
    tol = [0.0, 1e-9][k % 2 == 0 and k > 4]
    c, e, st = B.pow_simplify(dev(p.coef), dev(p.exps), k, tol, return_stats=True)
    assert st.key_bits == sum(int(k * int(mx)).bit_length() for mx in p.exps.max(axis=0))
    assert_parity(oracle_pow(p, k, tol), c.cpu().numpy(), e.cpu().numpy())


def test_power_of_a_wide_polynomial_and_the_table_path():
    """30 variables (p^3 needs 2 bits each... up to 8 bits: 240-bit keys): the packed intermediates are 256-bit keys; and a
    p_3^4 whose products (up to 6188 * 56 = 346,528) take the table path with packed output."""
    r = np.random.default_rng(5)
    p = W.Poly(r.standard_normal(40), r.integers(0, 80, size=(40, 30)).astype(np.uint8))
    c, e, st = B.pow_simplify(dev(p.coef), dev(p.exps), 3, 0.0, return_stats=True)
    assert st.key_bytes == 32
    assert_parity(oracle_pow(p, 3), c.cpu().numpy(), e.cpu().numpy())
    q = W.p_d(3)
    c, e, st = B.pow_simplify(dev(q.coef), dev(q.exps), 4, 0.0, return_stats=True, out_capacity=100_000)
    c, e = c.cpu().numpy(), e.cpu().numpy()
    assert len(c) == math.comb(5 + 12, 5) and c.sum() == float(56 ** 4) and (c == np.round(c)).all()
    assert st.table_path in (1, 2)

"""-m gpu: the one-block path (csrc/small.cu): at most 8192 (key, coefficient) pairs (4096 with 128-bit keys) are sorted
(radix sort of a permutation in shared memory) and summed by a single thread block, then pruned and unpacked -- the paper's
lightweight-operator regime (Table 7), where the multi-kernel path is all launch latency -- against the
CPU oracle."""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import assert_parity, dev

pytestmark = pytest.mark.gpu


def run(p, tol, flags=0, **kw):
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, flags=flags, **kw)
    torch.cuda.synchronize()
    return c.cpu().numpy(), e.cpu().numpy(), st


@pytest.mark.parametrize("n", [1, 2, 31, 33, 1000, 1024, 1025, 4097, 8191, 8192])
@pytest.mark.parametrize("shape", ["c1", "c5", "c3u"])
def test_small_inputs_match_the_oracle(n, shape):
    if shape == "c1":
        p, tol = W.config1(n)
    elif shape == "c5":
        p, tol = W.config5((n + 9) // 10 * 10)
        p = W.Poly(p.coef[:n], p.exps[:n])
    else:
        p, tol = W.config3u(n)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = run(p, tol)
    small = n <= (8192 if st.key_bytes == 8 else 4096)         # the keys must fit shared memory twice
    assert st.small_path == (1 if small else 0) and st.table_path == 0
    assert st.sort_passes == (0 if small else len(st.digit_bits))
    assert st.distinct == len(res.sum) and st.survivors == len(c)
    assert_parity(res, c, e)
    c0, e0, st0 = run(p, tol, flags=B.FLAG_NO_SMALL)
    assert st0.small_path == 0
    assert (e0 == e).all()
    # equal monomials are summed in input order on both paths up to the tree: same tolerance class, and here bit-identical
    # whenever every run lies inside one thread on both paths is not guaranteed -- compare under the parity rule only
    assert_parity(res, c0, e0)


def test_8193_terms_take_the_multi_kernel_path():
    p, tol = W.config1(8193)
    c, e, st = run(p, tol)
    assert st.small_path == 0
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


@pytest.mark.parametrize("n", [5, 3000, 8192])
def test_small_all_equal_and_all_distinct(n):
    r = np.random.default_rng(n)
    coef = r.standard_normal(n)
    exps = np.tile(np.array([[3, 1, 4, 1, 5]], np.uint8), (n, 1))
    c, e, st = run(W.Poly(coef, exps), 0.0)
    assert st.small_path == 1 and len(c) == 1
    assert abs(c[0] - float(np.sum(coef))) <= 1e-12 * np.abs(coef).sum()
    perm = r.permutation(n).astype(np.uint32)
    exps = np.stack([perm >> 8, perm & 0xff], axis=1).astype(np.uint16)
    c, e, st = run(W.Poly(coef, exps), 0.0)
    assert st.small_path == 1 and len(c) == n
    assert_parity(oracle.simplify(coef, exps, 0.0), c, e)
    # bit-reproducible, and a stable sort: the sums of a permuted input obey the parity rule
    c2, e2, _ = run(W.Poly(coef, exps), 0.0)
    assert (c.view(np.uint64) == c2.view(np.uint64)).all()


def test_small_tolerance_p_minus_p_capacity_and_dtypes():
    p, _ = W.config1(4000)
    coef = np.concatenate([p.coef, -p.coef])
    exps = np.concatenate([p.exps, p.exps])
    c, e, st = run(W.Poly(coef, exps), 1e-12)
    assert st.small_path == 1 and len(c) == 0                 # p - p is the zero polynomial (reading A3)
    exps2 = np.array([[1], [2], [3], [3]], np.uint8)
    c, e, _ = run(W.Poly(np.array([0.75, np.nextafter(0.75, 1.0), 0.5, 0.25]), exps2), 0.75)
    assert e.tolist() == [[2]] and c[0] == np.nextafter(0.75, 1.0)          # |s| == tol dropped, the next double kept (A2)
    nan = float("nan")
    c, e, _ = run(W.Poly(np.array([nan, 1.0, 2.0]), np.array([[1], [1], [2]], np.uint8)), 0.0)
    assert e.tolist() == [[2]] and c.tolist() == [2.0]        # NaN sums are dropped (A12)
    p, tol = W.config1(5000, dtype=np.uint32)
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p.coef), dev(p.exps), tol, out_capacity=10)
    assert ei.value.status == B.ERR_OUTPUT_TOO_SMALL
    c, e, st = run(p, tol)
    assert e.dtype == np.uint32 and st.small_path == 1
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


@pytest.mark.parametrize("na,nb", [(1, 1), (7, 5), (90, 91), (64, 128)])
def test_small_products(na, nb):
    r = np.random.default_rng(na * 1000 + nb)
    a = W.Poly(r.standard_normal(na), r.integers(0, 4, size=(na, 6)).astype(np.uint8))
    b = W.Poly(r.standard_normal(nb), r.integers(0, 4, size=(nb, 6)).astype(np.uint8))
    c, e, st = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), 0.0, return_stats=True)
    assert st.small_path == 1
    assert_parity(oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, 0.0), c.cpu().numpy(), e.cpu().numpy())


def test_small_async_device_count():
    """POLYLAB_FLAG_DEVICE_COUNT with caller bounds: three launches, no host synchronisation, count and status on the device."""
    p, tol = W.config1(6000)
    out_c = torch.empty(6000, dtype=torch.float64, device="cuda")
    out_e = torch.empty((6000, 4), dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    status = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    st = B.simplify_async(dev(p.coef), dev(p.exps), tol, [3, 3, 3, 3], out_c, out_e, cnt, status)
    torch.cuda.synchronize()
    k = int(cnt.item())
    assert int(status.item()) == 0 and k == 256
    assert_parity(oracle.simplify(p.coef, p.exps, tol), out_c[:k].cpu().numpy(), out_e[:k].cpu().numpy())

"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs -- paper examples, the five BASELINE.json configs at sizes the oracle finishes in seconds
(several tiles plus a ragged tail), stage-level checks, edge cases.  Rule: monomial set and exponents
bit-exact in canonical order, |gpu - oracle| <= 1e-12 * sum|contributions| (oracle/parity.py)."""
import json
import math
import os

import numpy as np
import pytest
import torch

from oracle import oracle, parity
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import assert_parity, check_mul, check_simplify, dev, gpu_mul, gpu_simplify

pytestmark = pytest.mark.gpu

with open(os.path.join(os.path.dirname(__file__), "golden", "paper_examples.json")) as f:
    PAPER = json.load(f)


# ------------------------------------------------------------------------------- paper examples

@pytest.mark.parametrize("dtype", [np.uint8, np.uint16, np.uint32])
@pytest.mark.parametrize("ex", PAPER["examples"], ids=[e["name"] for e in PAPER["examples"]])
def test_paper_examples(ex, dtype):
    if ex["op"] == "simplify":
        c, e = gpu_simplify(np.array(ex["coef"], float), np.array(ex["exps"], dtype), ex["tol"])
    else:
        a = W.Poly(np.array(ex["a_coef"], float), np.array(ex["a_exps"], dtype))
        b = W.Poly(np.array(ex["b_coef"], float), np.array(ex["b_exps"], dtype))
        c, e = gpu_mul(a, b, ex["tol"])
    assert e.dtype == dtype
    got = {tuple(int(x) for x in r): float(v) for v, r in zip(c, e)}
    want = {tuple(r): float(v) for v, r in zip(ex["out_coef"], ex["out_exps"])}
    assert got == want, ex["cite"]
    assert e.tolist() == sorted(e.tolist())
    if ex["ordered"]:
        assert e.tolist() == ex["out_exps"] and c.tolist() == [float(v) for v in ex["out_coef"]], ex["cite"]


@pytest.mark.parametrize("n,k", [(2, 6), (3, 5), (5, 4), (8, 4)])
def test_multinomial_closed_form_gpu(n, k):
    """(x1+...+xn)^k by chained mul_simplify: C(n+k-1,k) terms, multinomial coefficients, bit-exact."""
    base = W.Poly(np.ones(n), np.eye(n, dtype=np.uint8))
    c, e = base.coef, base.exps
    for _ in range(k - 1):
        c, e = gpu_mul(W.Poly(c, e), base)
    assert len(c) == math.comb(n + k - 1, k)
    for coef, row in zip(c, e.tolist()):
        want = math.factorial(k)
        for x in row:
            want //= math.factorial(x)
        assert coef == float(want)


@pytest.mark.parametrize("d", [2, 3, 4])
def test_paper_pd_cubed_gpu(d):
    """The paper's Fig. 2 workload simplify(p_d^3), 5 variables: C(5+3d,5) terms,
    integer coefficients summing to C(5+d,d)^3; chained and one-shot expansion agree exactly."""
    p = W.p_d(d)
    c2, e2 = gpu_mul(p, p)
    assert len(c2) == math.comb(5 + 2 * d, 5)
    c3, e3 = gpu_mul(W.Poly(c2, e2), p)
    assert len(c3) == math.comb(5 + 3 * d, 5)
    assert c3.sum() == float(p.nterms ** 3) and (c3 == np.round(c3)).all() and c3.min() >= 1.0
    # one shot: raw p*p (not merged), times p
    rc, re_ = B.expand(dev(p.coef), dev(p.exps), dev(p.coef), dev(p.exps))
    assert rc.shape[0] == p.nterms ** 2
    c1, e1 = B.mul_simplify(rc, re_, dev(p.coef), dev(p.exps))
    assert e1.cpu().numpy().tolist() == e3.tolist() and c1.cpu().numpy().tolist() == c3.tolist()
    if d <= 3:
        res = oracle.mul_simplify(c2, e2, p.coef, p.exps)
        assert_parity(res, c3, e3)
        assert res.sum.tolist() == c3.tolist()


# ------------------------------------------------------------------------------- stage S1 alone

def _lex_order(exps):
    return np.lexsort(exps[:, ::-1].T.astype(np.int64))      # stable; column 0 most significant


@pytest.mark.parametrize("case", ["c1", "c3", "c4", "c5", "u16", "u32wide", "bits128", "colmajor"])
def test_pack_keys_order_is_lexicographic(case):
    r = np.random.default_rng(42)
    kw = {}
    if case == "c1":
        exps = W.config1(20_000)[0].exps
    elif case == "c3":
        exps = W.config3(20_000)[0].exps
    elif case == "c4":
        exps = W.config4(200)[0].exps
    elif case == "c5":
        exps = W.config5(20_000)[0].exps
    elif case == "u16":
        exps = W.config3u(20_000)[0].exps
    elif case == "u32wide":
        exps = r.integers(0, 2 ** 32, size=(5000, 4), dtype=np.uint64).astype(np.uint32)
        exps[:, 1] = r.integers(0, 3, 5000)             # narrow field between wide ones; straddles bit 64
    elif case == "bits128":
        exps = r.integers(0, 2, size=(5000, 128)).astype(np.uint8)
    else:
        exps = W.config5(10_000)[0].exps
    t = dev(exps)
    if case == "colmajor":
        t = dev(np.asfortranarray(exps).T.copy()).T          # same values, column-major storage (MATLAB pow)
        assert not t.is_contiguous()
    keys, bits = B.pack_keys(t, **kw)
    keys = keys.cpu().numpy().view(np.uint64)
    want_bits = sum(int(m).bit_length() for m in exps.max(axis=0))
    assert bits == want_bits
    order_keys = np.lexsort((keys[:, 1], keys[:, 0]))
    order_rows = _lex_order(exps)
    assert (order_keys == order_rows).all()
    # equal keys <=> equal rows (checked on the sorted sequence)
    ks, rs = keys[order_keys], exps[order_rows]
    same_k = (ks[1:] == ks[:-1]).all(axis=1)
    same_r = (rs[1:] == rs[:-1]).all(axis=1)
    assert (same_k == same_r).all()
    if want_bits <= 64:
        assert (keys[:, 0] == 0).all()


# ------------------------------------------------------------------------------- the five configs

def test_config1_full():
    p, tol = W.config1()
    rep, (c, e), res = check_simplify(p.coef, p.exps, tol)
    assert len(c) == 256 and rep.matched == 256


@pytest.mark.parametrize("dtype", [np.uint8, np.uint32])
@pytest.mark.parametrize("n", [1, 31, 4097, 50_001])
def test_config1_sizes(n, dtype):
    p, tol = W.config1(n, dtype=dtype)
    check_simplify(p.coef, p.exps, tol)


@pytest.mark.parametrize("n_each", [37, 300, 2000])
def test_config2(n_each):
    a, b, tol = W.config2(n_each)
    rep, (c, e), res = check_mul(a, b, tol)
    assert rep.matched == res.keep.sum()


@pytest.mark.parametrize("n", [10_000, 1_000_003])
def test_config3(n):
    p, tol = W.config3(n)
    rep, (c, e), _ = check_simplify(p.coef, p.exps, tol)
    assert len(c) <= 7680


def test_config3u_mostly_unique_128bit():
    p, tol = W.config3u(300_001)
    rep, (c, e), res = check_simplify(p.coef, p.exps, tol)
    assert len(c) > 299_000 and e.dtype == np.uint16


def test_config4_cubic_both_variants():
    """Two chained mul+simplify passes (variant A) and the 8e6-term one-shot second pass (variant B, A16);
    checked against the oracle, against each other and by evaluation at 16 random points (A19)."""
    p, tol = W.config4()
    cq, eq = gpu_mul(p, p, tol)
    res_q = oracle.mul_simplify(p.coef, p.exps, p.coef, p.exps, tol)
    assert_parity(res_q, cq, eq)
    ca, ea = gpu_mul(W.Poly(cq, eq), p, tol)
    res_a = oracle.mul_simplify(cq, eq, p.coef, p.exps, tol)
    assert_parity(res_a, ca, ea)
    # variant B: raw 40,000-term p*p, then times p = 8e6 products in one sort
    rc, re_ = B.expand(dev(p.coef), dev(p.exps), dev(p.coef), dev(p.exps))
    assert rc.shape[0] == 40_000
    cb, eb, st = B.mul_simplify(rc, re_, dev(p.coef), dev(p.exps), tol, return_stats=True)
    assert st.sort_terms == 8_000_000 and 40 <= st.key_bits <= 60 and st.key_bytes == 8
    cb, eb = cb.cpu().numpy(), eb.cpu().numpy()
    assert eb.tolist() == ea.tolist()
    # A vs B differ only in summation order
    absum = oracle.simplify(np.abs(np.concatenate([ca, cb])), np.concatenate([ea, eb])).sum
    assert (np.abs(ca - cb) <= 1e-12 * np.maximum(absum, 1e-300) * 200).all()
    for x in W.eval_points(20, 16):
        px, _ = oracle.evaluate(p.coef, p.exps, x)
        for (c, e) in ((ca, ea), (cb, eb)):
            rx, ra = oracle.evaluate(c, e, x)
            assert abs(rx - px ** 3) <= 1e-10 * ra + 1e-300


@pytest.mark.parametrize("n", [10_000, 1_000_000])
def test_config5(n):
    p, tol = W.config5(n)
    rep, (c, e), res = check_simplify(p.coef, p.exps, tol)
    assert len(res.sum) == n // 10
    assert len(c) == n // 20           # the cancelling half is pruned exactly (A18)


# ------------------------------------------------------------------------------- edge cases

def test_empty_and_single():
    c, e = gpu_simplify(np.zeros(0), np.zeros((0, 3), np.uint8))
    assert c.shape == (0,) and e.shape == (0, 3)
    c, e = gpu_simplify(np.array([2.5]), np.array([[7, 0, 9]], np.uint8))
    assert c.tolist() == [2.5] and e.tolist() == [[7, 0, 9]]
    c, e = gpu_simplify(np.array([0.0]), np.array([[7, 0, 9]], np.uint8))
    assert len(c) == 0
    a = W.Poly(np.zeros(0), np.zeros((0, 3), np.uint8))
    b = W.Poly(np.ones(2), np.ones((2, 3), np.uint8))
    c, e = gpu_mul(a, b)
    assert len(c) == 0


@pytest.mark.parametrize("n", [5, 2304, 2305, 60_000])
def test_all_equal_keys_one_run_spanning_tiles(n):
    r = np.random.default_rng(n)
    coef = r.standard_normal(n)
    exps = np.tile(np.array([[3, 1, 4, 1, 5]], np.uint8), (n, 1))
    rep, (c, e), res = check_simplify(coef, exps)
    assert len(c) == 1 and abs(c[0] - math.fsum(coef.tolist())) <= 1e-12 * np.abs(coef).sum()


def test_all_zero_exponents_no_sort_pass():
    coef = np.arange(1, 5001, dtype=float)
    exps = np.zeros((5000, 6), np.uint8)
    c, e, st = B.simplify(dev(coef), dev(exps), return_stats=True)
    assert st.key_bits == 0 and st.sort_passes == 0
    assert c.cpu().tolist() == [float(5000 * 5001 // 2)] and e.cpu().tolist() == [[0] * 6]


@pytest.mark.parametrize("n", [4096, 100_003])
def test_all_distinct(n):
    r = np.random.default_rng(1)
    perm = r.permutation(n).astype(np.uint32)
    exps = np.stack([perm >> 12, perm & 0xfff, np.zeros(n, np.uint32)], axis=1).astype(np.uint16)
    coef = r.standard_normal(n)
    rep, (c, e), _ = check_simplify(coef, exps)
    assert len(c) == n
    order = np.argsort(perm)
    assert (c == coef[order]).all()          # single contributions: bit-exact


def test_runs_crossing_every_tile_boundary():
    """Runs of 1000 equal keys over 100 keys: segments straddle reduce tiles (2304) and sort tiles."""
    r = np.random.default_rng(3)
    n = 100_000
    key = np.repeat(np.arange(100, dtype=np.uint8), 1000)
    exps = np.stack([key, 255 - key], axis=1)
    coef = r.standard_normal(n)
    perm = r.permutation(n)
    check_simplify(coef[perm], exps[perm])
    check_simplify(coef, exps)               # already sorted input


def test_p_minus_p_is_zero_polynomial():
    """Invariant p - p = 0 (north_star).  At tol = 0 floating-point residues of a reordered sum may survive;
    they lie inside the rule's exemption band.  At any tol above the rounding level the result is empty."""
    p, _ = W.config3(200_000)
    coef = np.concatenate([p.coef, -p.coef])
    exps = np.concatenate([p.exps, p.exps])
    perm = np.random.default_rng(0).permutation(len(coef))
    c, e = gpu_simplify(coef[perm], exps[perm], 0.0)
    res = oracle.simplify(coef[perm], exps[perm], 0.0)
    assert res.keep.sum() == 0
    rep = assert_parity(res, c, e)
    assert rep.exempt == len(res.sum)
    c, e = gpu_simplify(coef[perm], exps[perm], 1e-12)
    assert len(c) == 0
    # integer coefficients cancel exactly in any order: the zero polynomial at tol = 0
    ci = np.round(p.coef * 1024)
    c, e = gpu_simplify(np.concatenate([ci, -ci])[perm], exps[perm], 0.0)
    assert len(c) == 0


def test_tolerance_semantics_gpu():
    tol = 0.25
    up = math.nextafter(tol, 1.0)
    coef = np.array([0.25, -0.25, up, -up, 0.125, 0.125, 0.1, 100.0, 1.0, -1.0, float("nan")])
    exps = np.array([[0], [1], [2], [3], [4], [4], [5], [5], [6], [6], [7]], np.uint8)
    c, e = gpu_simplify(coef, exps, tol)
    assert e[:, 0].tolist() == [2, 3, 5] and c.tolist() == [up, -up, 100.1]
    c, e = gpu_simplify(np.array([-0.0, 5e-324, 1.0, -1.0]), np.array([[0], [1], [2], [2]], np.uint8), 0.0)
    assert e[:, 0].tolist() == [1] and c.tolist() == [5e-324]


def test_nonfinite_coefficients_gpu():
    """Reading A12 on both sides: +-inf sums are kept, inf - inf and NaN sums are dropped."""
    inf = float("inf")
    coef = np.array([inf, 1.0, 2.0, -inf, 3.0, inf, -inf, 4.0, 1.5, float("nan"), 7.0])
    exps = np.array([[0], [0], [1], [1], [1], [2], [2], [2], [3], [4], [4]], np.uint8)
    c, e = gpu_simplify(coef, exps, 0.5)
    assert e[:, 0].tolist() == [0, 1, 3] and c.tolist() == [inf, -inf, 1.5]
    res = oracle.simplify(coef, exps, 0.5)
    assert res.pruned[0].tolist() == c.tolist() and res.pruned[1][:, 0].tolist() == e[:, 0].tolist()


def test_strides_column_major_and_dtypes():
    p, tol = W.config3(50_000)
    res = oracle.simplify(p.coef, p.exps, tol)
    for dt, tdt in ((np.uint8, torch.uint8), (np.uint16, torch.uint16), (np.uint32, torch.uint32)):
        ex = p.exps.astype(dt)
        c, e = gpu_simplify(p.coef, ex, tol)
        assert_parity(res, c, e)
        colmajor = dev(np.ascontiguousarray(ex.T)).T          # element (t,v) at t*1 + v*nterms
        assert colmajor.stride() == (1, 50_000)
        c2, e2 = B.simplify(dev(p.coef), colmajor, tol)
        assert e2.dtype == tdt and (e2.cpu().numpy() == e).all() and (c2.cpu().numpy() == c).all()
    # unaligned base pointer: generic strided kernel
    big = dev(np.concatenate([np.zeros((1, 10), np.uint8), p.exps]))
    c3, e3 = B.simplify(dev(p.coef), big[1:], tol)
    assert (e3.cpu().numpy() == e.astype(np.uint8)).all()


def test_caller_bounds_and_errors():
    p, tol = W.config1(30_000)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), tol, max_exp=[3, 3, 3, 3], return_stats=True)
    assert_parity(res, c.cpu().numpy(), e.cpu().numpy())
    assert st.key_bits == 8 and st.sort_passes == 1
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), tol, max_exp=[7, 3, 200, 3], return_stats=True)   # loose bounds
    assert_parity(res, c.cpu().numpy(), e.cpu().numpy())
    assert st.key_bits == 3 + 2 + 8 + 2
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p.coef), dev(p.exps), tol, max_exp=[3, 3, 2, 3])
    assert ei.value.status == B.ERR_EXPONENT_RANGE
    wide = np.full((10, 33), 255, np.uint8)                # 264 bits: one more than four words hold
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(np.ones(10)), dev(wide))
    assert ei.value.status == B.ERR_KEY_TOO_WIDE
    with pytest.raises(B.PolylabError) as ei:      # 200 + 100 does not fit uint8
        B.mul_simplify(dev(np.ones(1)), dev(np.array([[200]], np.uint8)), dev(np.ones(1)), dev(np.array([[100]], np.uint8)))
    assert ei.value.status == B.ERR_EXPONENT_RANGE
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p.coef), dev(p.exps), tol, out_capacity=100)
    assert ei.value.status == B.ERR_OUTPUT_TOO_SMALL


def test_128_one_bit_variables_and_wide_fields():
    r = np.random.default_rng(9)
    exps = r.integers(0, 2, size=(20_000, 128)).astype(np.uint8)
    exps[:, 5:120] = 0
    exps[::2] = exps[1::2]                  # force duplicates
    coef = r.standard_normal(20_000)
    c, e, st = B.simplify(dev(coef), dev(exps), return_stats=True)
    assert st.key_bits <= 13
    assert_parity(oracle.simplify(coef, exps), c.cpu().numpy(), e.cpu().numpy())
    full = r.integers(0, 2, size=(3000, 128)).astype(np.uint8)
    full[:, :] |= (np.arange(128) % 2 == 0).astype(np.uint8) & full           # keep all 128 fields live
    coef = r.standard_normal(3000)
    c, e, st = B.simplify(dev(coef), dev(full), return_stats=True)
    assert st.key_bits == 128 and st.key_bytes == 16 and len(st.digit_bits) == 16
    assert_parity(oracle.simplify(coef, full), c.cpu().numpy(), e.cpu().numpy())
    big = r.integers(0, 2 ** 32, size=(4000, 3), dtype=np.uint64).astype(np.uint32)
    big[0:3999:3] = big[1:4000:3]
    coef = r.standard_normal(4000)
    c, e, st = B.simplify(dev(coef), dev(big), return_stats=True)
    assert st.key_bits == 96
    assert_parity(oracle.simplify(coef, big), c.cpu().numpy(), e.cpu().numpy())


def test_bit_reproducible_and_permutation_invariant():
    p, tol = W.config5(200_000)
    c1, e1 = gpu_simplify(p.coef, p.exps, tol)
    c2, e2 = gpu_simplify(p.coef, p.exps, tol)
    assert (e1 == e2).all() and (c1.view(np.uint64) == c2.view(np.uint64)).all()
    perm = np.random.default_rng(1).permutation(p.nterms)
    c3, e3 = gpu_simplify(p.coef[perm], p.exps[perm], tol)
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c3, e3)
    # idempotence: simplify(simplify(p)) == simplify(p) bit-exact
    c4, e4 = gpu_simplify(c1, e1, tol)
    assert (e4 == e1).all() and (c4.view(np.uint64) == c1.view(np.uint64)).all()
    # scaling by a power of two scales the result exactly
    c5, _ = gpu_simplify(p.coef * 2.0 ** 20, p.exps, tol * 2.0 ** 20)
    assert (c5 == c1 * 2.0 ** 20).all()


def test_expand_raw_matches_oracle_exactly():
    a, b, _ = W.config2(150)
    rc, re_ = B.expand(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps))
    oc, orow = oracle.expand(a.coef, a.exps, b.coef, b.exps)
    assert (rc.cpu().numpy().view(np.uint64) == oc.view(np.uint64)).all()      # one IEEE multiplication each
    assert (re_.cpu().numpy() == orow).all()


def test_product_commutes_and_evaluates():
    a, b, tol = W.config2(400)
    c1, e1 = gpu_mul(a, b, tol)
    c2, e2 = gpu_mul(b, a, tol)
    assert (e1 == e2).all()
    res = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol)
    assert_parity(res, c2, e2)
    for x in W.eval_points(6, 4):
        va, _ = oracle.evaluate(a.coef, a.exps, x)
        vb, _ = oracle.evaluate(b.coef, b.exps, x)
        vr, ar = oracle.evaluate(c1, e1, x)
        assert abs(vr - va * vb) <= 1e-11 * ar


def test_host_entry_points():
    p, tol = W.config5(100_000)
    c, e, st = B.simplify_host(p.coef, p.exps, tol, return_stats=True)
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)
    assert st.key_bytes == 16 and st.kernel_launches >= 19
    a, b, tol = W.config2(200)
    c, e = B.mul_simplify_host(a.coef, a.exps, b.coef, b.exps, tol)
    assert_parity(oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol), c, e)
    # pinned host tensors in and out
    pc, pe = torch.from_numpy(p.coef).pin_memory(), torch.from_numpy(p.exps).pin_memory()
    oc, oe = torch.empty(p.nterms, dtype=torch.float64).pin_memory(), torch.empty((p.nterms, 16), dtype=torch.uint8).pin_memory()
    c2, e2 = B.simplify_host(pc, pe, 1e-14, out=(oc, oe))
    assert_parity(oracle.simplify(p.coef, p.exps, 1e-14), c2.numpy(), e2.numpy())


def test_async_device_count():
    p, tol = W.config1(50_000)
    n = p.nterms
    oc = torch.empty(n, dtype=torch.float64, device="cuda")
    oe = torch.empty((n, 4), dtype=torch.uint8, device="cuda")
    cnt = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    status = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    B.simplify_async(dev(p.coef), dev(p.exps), tol, [3, 3, 3, 3], oc, oe, cnt, status)
    torch.cuda.synchronize()
    k = int(cnt.item())
    assert int(status.item()) == 0 and k == 256
    assert_parity(oracle.simplify(p.coef, p.exps, tol), oc[:k].cpu().numpy(), oe[:k].cpu().numpy())


# ------------------------------------------------------------------------------- ranking kernels

@pytest.mark.parametrize("cfg", ["c3", "c5", "c2"])
def test_safe_rank_kernel_matches_default(cfg):
    """The ballot-matching radix pass (POLYLAB_FLAG_SAFE_RANK) and the default atomic-ranking pass are both stable:
    same monomials, bit-identical sums (the summation tree is the same when the sorted order is the same)."""
    if cfg == "c2":
        a, b, tol = W.config2(300)
        r0 = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, return_stats=True, flags=B.FLAG_NO_TABLE)
        r1 = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, return_stats=True, flags=B.FLAG_SAFE_RANK)
        res = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol)
    else:
        p, tol = (W.config3(300_000) if cfg == "c3" else W.config5(300_000))
        r0 = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, flags=B.FLAG_NO_TABLE)    # the sort path
        r1 = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, flags=B.FLAG_SAFE_RANK)
        res = oracle.simplify(p.coef, p.exps, tol)
    assert r0[2].rank_fallback == 0 and r1[2].rank_fallback == 0
    c0, e0, c1, e1 = r0[0].cpu().numpy(), r0[1].cpu().numpy(), r1[0].cpu().numpy(), r1[1].cpu().numpy()
    assert_parity(res, c0, e0)
    assert (e0 == e1).all() and (c0.view(np.uint64) == c1.view(np.uint64)).all()


def test_unstable_rank_is_detected_and_falls_back():
    """POLYLAB_FLAG_DEBUG_UNSTABLE reverses the lane order of the atomic-ranking pass, which breaks LSD stability;
    the segmented-sum step must see the unsorted keys and the call must re-run with the ballot kernel."""
    p, tol = W.config5(300_000)
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, flags=B.FLAG_DEBUG_UNSTABLE)
    assert st.rank_fallback == 1
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c.cpu().numpy(), e.cpu().numpy())
    a, b, tol = W.config2(300)
    c, e, st = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, return_stats=True,
                              flags=B.FLAG_DEBUG_UNSTABLE)
    assert st.rank_fallback == 1
    assert_parity(oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol), c.cpu().numpy(), e.cpu().numpy())


@pytest.mark.parametrize("shape", ["c2", "c4sq", "wide128", "tiny"])
def test_fused_expand_matches_materialised_products(shape):
    """X1 runs inside the first radix pass by default (products formed in registers, never stored); with
    POLYLAB_FLAG_NO_FUSED_PACK the products are materialised first.  Same order of records -> bit-identical results."""
    r = np.random.default_rng(77)
    if shape == "c2":
        a, b, tol = W.config2(700)
    elif shape == "c4sq":
        p, tol = W.config4()
        a, b = p, p
    elif shape == "wide128":
        a = W.Poly(r.standard_normal(900), r.integers(0, 100, size=(900, 12)).astype(np.uint8))
        b = W.Poly(r.standard_normal(40), r.integers(0, 100, size=(40, 12)).astype(np.uint8))
        tol = 0.0
    else:
        a = W.Poly(np.array([1.0, 2.0]), np.array([[1, 0], [0, 1]], np.uint8))
        b = W.Poly(np.array([1.0, -2.0]), np.array([[1, 0], [0, 1]], np.uint8))
        tol = 0.0
    r0 = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, return_stats=True, flags=B.FLAG_NO_TABLE)
    r1 = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, return_stats=True,
                        flags=B.FLAG_NO_FUSED_PACK | B.FLAG_NO_TABLE)
    c0, e0, c1, e1 = r0[0].cpu().numpy(), r0[1].cpu().numpy(), r1[0].cpu().numpy(), r1[1].cpu().numpy()
    assert (e0 == e1).all() and (c0.view(np.uint64) == c1.view(np.uint64)).all()
    assert r0[2].kernel_launches == r1[2].kernel_launches
    assert_parity(oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol), c0, e0)


@pytest.mark.parametrize("seed", range(24))
def test_randomised_products_all_paths(seed):
    """Random operand sizes, variable counts, dtypes and exponent ranges: the default product path (X1 fused into the
    first pass), the materialising path, the forced bucket path and the ballot-ranking path all in parity with the oracle."""
    r = np.random.default_rng(70_000 + seed)
    dtype = [np.uint8, np.uint16, np.uint32][int(r.integers(0, 3))]
    nvars = int(r.integers(1, 13))
    hi = int(r.choice([2, 4, 16, 100]))
    na, nb = int(r.choice([1, 7, 200, 1100])), int(r.choice([1, 5, 64, 1100]))
    a = W.Poly(r.standard_normal(na), r.integers(0, hi, size=(na, nvars)).astype(dtype))
    b = W.Poly(r.standard_normal(nb), r.integers(0, hi, size=(nb, nvars)).astype(dtype))
    tol = [0.0, 1e-13][seed % 2]
    res = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol)
    for flags in (0, B.FLAG_NO_TABLE, B.FLAG_DEBUG_FORCE_TABLE, B.FLAG_DEBUG_FORCE_TABLE | B.FLAG_DEBUG_FORCE_HASH,
                  B.FLAG_DEBUG_FORCE_BUCKET, B.FLAG_NO_FUSED_PACK | B.FLAG_NO_TABLE, B.FLAG_SAFE_RANK):
        c, e = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, flags=flags)
        assert_parity(res, c.cpu().numpy(), e.cpu().numpy())

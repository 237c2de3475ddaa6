"""-m gpu: batched simplify and the polynomial-matrix product (csrc/batch.cu) against the CPU oracle called
once per entry: polynomial matrices are arrays of scalar polynomials and mtimes / sum apply the scalar operations entry
by entry (Table 4; section 3.4, with the worked example A^2 for A = [x1 1; 0 x2])."""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import assert_parity, dev

pytestmark = pytest.mark.gpu


def random_matrix(r, rows, cols, nvars, max_terms, hi, dtype=np.uint8, empty_prob=0.15):
    """rows*cols random scalar polynomials (row-major), some of them empty: (coef, exps, offsets)."""
    coefs, exps, off = [], [], [0]
    for _ in range(rows * cols):
        nt = 0 if r.random() < empty_prob else int(r.integers(1, max_terms + 1))
        coefs.append(r.standard_normal(nt))
        exps.append(r.integers(0, hi, size=(nt, nvars)).astype(dtype))
        off.append(off[-1] + nt)
    return np.concatenate(coefs), np.concatenate(exps).reshape(-1, nvars).astype(dtype), np.array(off, np.int64)


def entry(c, e, off, idx):
    return c[off[idx]:off[idx + 1]], e[off[idx]:off[idx + 1]]


def oracle_matmul_entry(A, B_, m, k, n, i, j, tol):
    """sum over l of A(i,l)*B(l,j): the raw products of every l concatenated, then ONE oracle simplify."""
    cs, es = [], []
    nvars = A[1].shape[1]
    for l in range(k):
        ca, ea = entry(*A, i * k + l)
        cb, eb = entry(*B_, l * n + j)
        if len(ca) and len(cb):
            c, e = oracle.expand(ca, ea, cb, eb)
            cs.append(c)
            es.append(e)
    if not cs:
        return oracle.simplify(np.zeros(0), np.zeros((0, nvars), np.uint32), tol)
    return oracle.simplify(np.concatenate(cs), np.concatenate(es), tol)


def test_paper_matrix_square_example():
    """A = [x1 1; 0 x2]: A^2 = [x1^2, x1 + x2; 0, x2^2]."""
    coef = np.array([1.0, 1.0, 1.0])                   # entries: (x1), (1), (), (x2)
    exps = np.array([[1, 0], [0, 0], [0, 1]], np.uint8)
    off = np.array([0, 1, 2, 2, 3], np.int64)
    c, e, o = B.matmul_simplify(dev(coef), dev(exps), off, dev(coef), dev(exps), off, 2, 2, 2)
    c, e = c.cpu().numpy(), e.cpu().numpy()
    assert o.tolist() == [0, 1, 3, 3, 4]
    assert e.tolist() == [[2, 0], [0, 1], [1, 0], [0, 2]] and c.tolist() == [1.0, 1.0, 1.0, 1.0]


@pytest.mark.parametrize("seed,m,k,n,nvars,max_terms,hi,dtype", [
    (0, 3, 3, 3, 3, 12, 4, np.uint8),          # the 3x3 case: 9 entries x 3 products each
    (1, 2, 5, 4, 6, 30, 3, np.uint8),
    (2, 1, 1, 1, 2, 60, 5, np.uint16),
    (3, 4, 2, 3, 20, 9, 8, np.uint8),          # 60 + 4 bits: one 64-bit word
    (4, 3, 3, 3, 12, 40, 200, np.uint8),       # 192 bits would not fit: 12 variables x 9 bits + entry = 128-bit keys
    (5, 6, 6, 6, 5, 25, 4, np.uint32),         # ~1e5 products: the multi-kernel LSD tail
])
def test_matrix_product_matches_one_oracle_call_per_entry(seed, m, k, n, nvars, max_terms, hi, dtype):
    r = np.random.default_rng(500 + seed)
    hi2 = min(hi, 120) if dtype == np.uint8 else hi                     # sums must fit the dtype
    A = random_matrix(r, m, k, nvars, max_terms, hi2, dtype)
    B_ = random_matrix(r, k, n, nvars, max_terms, hi2, dtype)
    tol = [0.0, 1e-13][seed % 2]
    c, e, o, st = B.matmul_simplify(dev(A[0]), dev(A[1]), A[2], dev(B_[0]), dev(B_[1]), B_[2], m, k, n, tol, return_stats=True)
    c, e = c.cpu().numpy(), e.cpu().numpy()
    assert o[0] == 0 and len(o) == m * n + 1 and o[-1] == len(c) and (np.diff(o) >= 0).all()
    for i in range(m):
        for j in range(n):
            res = oracle_matmul_entry(A, B_, m, k, n, i, j, tol)
            ce, ee = entry(c, e, o, i * n + j)
            assert_parity(res, ce, ee)
    # the same through separate calls: per entry, raw products (polylab_expand) concatenated and simplified
    for (i, j) in [(0, 0), (m - 1, n - 1)]:
        cs, es = [], []
        for l in range(k):
            ca, ea = entry(*A, i * k + l)
            cb, eb = entry(*B_, l * n + j)
            if len(ca) and len(cb):
                pc, pe = B.expand(dev(ca), dev(ea), dev(cb), dev(eb))
                cs.append(pc)
                es.append(pe)
        ce, ee = entry(c, e, o, i * n + j)
        if cs:
            c1, e1 = B.simplify(torch.cat(cs), torch.cat(es), tol)
            assert (e1.cpu().numpy() == ee).all()
        else:
            assert len(ce) == 0


def test_simplify_batched_matches_one_oracle_call_per_entry():
    r = np.random.default_rng(42)
    c, e, off = random_matrix(r, 3, 3, 4, 400, 3)                       # heavy duplication inside every entry
    gc, ge, go, st = B.simplify_batched(dev(c), dev(e), off, 0.0, return_stats=True)
    gc, ge = gc.cpu().numpy(), ge.cpu().numpy()
    assert st.small_path == 1
    for k in range(9):
        ce, ee = entry(c, e, off, k)
        assert_parity(oracle.simplify(ce, ee, 0.0), *entry(gc, ge, go, k))
    # a larger batch: 300 polynomials, 2e5 terms -> LSD tail; p - p entries vanish (zero polynomial: equal offsets, A3)
    c, e, off = random_matrix(r, 30, 10, 5, 1300, 6, empty_prob=0.05)
    t0, t1 = off[7], off[8]
    half = (t1 - t0) // 2
    c[t0 + half:t0 + 2 * half] = -c[t0:t0 + half]
    e[t0 + half:t0 + 2 * half] = e[t0:t0 + half]
    if (t1 - t0) % 2:
        c[t1 - 1] = 0.0
    gc, ge, go, st = B.simplify_batched(dev(c), dev(e), off, 1e-12, return_stats=True)
    gc, ge = gc.cpu().numpy(), ge.cpu().numpy()
    assert st.small_path == 0 and go[8] == go[7]
    for k in range(300):
        ce, ee = entry(c, e, off, k)
        assert_parity(oracle.simplify(ce, ee, 1e-12), *entry(gc, ge, go, k))


def test_batched_sum_along_a_dimension():
    """sum(A, 2) of a polynomial matrix: lay each row's entries back to back -> one entry per row."""
    r = np.random.default_rng(7)
    c, e, off = random_matrix(r, 4, 6, 3, 20, 3, empty_prob=0.0)
    row_off = off[::6]
    gc, ge, go = B.simplify_batched(dev(c), dev(e), row_off, 0.0)
    gc, ge = gc.cpu().numpy(), ge.cpu().numpy()
    for i in range(4):
        assert_parity(oracle.simplify(c[row_off[i]:row_off[i + 1]], e[row_off[i]:row_off[i + 1]], 0.0), *entry(gc, ge, go, i))


def test_batched_errors_and_edges():
    c, e, off = np.ones(3), np.array([[200], [100], [1]], np.uint8), np.array([0, 1, 2, 3], np.int64)
    # empty batch / all entries empty
    gc, ge, go = B.simplify_batched(dev(np.zeros(0)), dev(np.zeros((0, 2), np.uint8)), np.array([0, 0, 0], np.int64))
    assert len(gc) == 0 and go.tolist() == [0, 0, 0]
    # a product whose exponent sum does not fit u8
    with pytest.raises(B.PolylabError) as ei:
        B.matmul_simplify(dev(c[:1]), dev(e[:1]), off[:2], dev(c[1:2]), dev(e[1:2]), off[:2], 1, 1, 1)
    assert ei.value.status == B.ERR_EXPONENT_RANGE
    # capacity
    r = np.random.default_rng(1)
    c, e, off = random_matrix(r, 2, 2, 3, 50, 4, empty_prob=0.0)
    with pytest.raises(B.PolylabError) as ei:
        B.simplify_batched(dev(c), dev(e), off, 0.0, out_capacity=3)
    assert ei.value.status == B.ERR_OUTPUT_TOO_SMALL
    # shape mismatch
    with pytest.raises(B.PolylabError):
        B.matmul_simplify(dev(c), dev(e), off, dev(c), dev(e), off, 2, 2, 3)

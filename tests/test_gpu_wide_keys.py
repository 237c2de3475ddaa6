"""-m gpu: keys of three and four 64-bit words ("multi-word for wide variable sets"; the paper's wide case is
the 500-variable sparse quartic family of PAPER.md:546).  129..256 key bits travel as a 256-bit key through the same
pack / radix sort / segmented sum / prune / unpack kernels (and the one-block path, products, batches); wider keys are
POLYLAB_ERR_KEY_TOO_WIDE.  Everything against the CPU oracle, which has no keys at all."""
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


def pooled(n, nvars, dup, seed, hi=256, dtype=np.uint8):
    r = np.random.default_rng(seed)
    pool = r.integers(0, hi, size=(max(1, n // dup), nvars)).astype(dtype)
    exps = pool[r.integers(0, len(pool), size=n)]
    return W.Poly(r.standard_normal(n), np.ascontiguousarray(exps))


@pytest.mark.parametrize("n", [1, 700, 2048, 2049, 30_001, 400_003])
def test_192_bit_keys(n):
    """24 variables of 8 bits: three words.  Small n: the one-block path (2048 pairs of 256-bit keys); else 24 LSD passes."""
    p = pooled(n, 24, 5, seed=n)
    c, e, st = run(p, 0.0)
    assert st.key_bits == (192 if n > 100 else st.key_bits) and st.key_bytes == (32 if st.key_bits > 128 else st.key_bytes)
    if n > 100:
        assert len(st.digit_bits) == 24 and st.small_path == (1 if n <= 2048 else 0) and st.prefix_passes == 0 and st.table_path == 0
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)
    c2, e2, _ = run(p, 0.0, flags=B.FLAG_SAFE_RANK)                   # the ballot-ranking kernel
    assert (e2 == e).all()
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c2, e2)


def test_200_one_bit_variables():
    r = np.random.default_rng(9)
    n = 20_000
    exps = r.integers(0, 2, size=(n, 200)).astype(np.uint8)
    exps[:, 3:190] &= (r.random((1, 187)) < 0.5).astype(np.uint8)   # about half of the variables are identically zero
    exps[::2] = exps[1::2]                                          # duplicates
    coef = r.standard_normal(n)
    c, e, st = run(W.Poly(coef, exps), 0.0)
    assert 64 < st.key_bits <= 200
    assert_parity(oracle.simplify(coef, exps), c, e)
    full = r.integers(0, 2, size=(6000, 200)).astype(np.uint8)
    full[:200] |= np.eye(200, dtype=np.uint8)                       # every field live: 200 key bits, four words
    full[3000:] = full[:3000]
    coef = r.standard_normal(6000)
    c, e, st = run(W.Poly(coef, full), 0.0)
    assert st.key_bits == 200 and st.key_bytes == 32 and len(st.digit_bits) == 25
    assert_parity(oracle.simplify(coef, full), c, e)
    assert len(c) <= 3000


def test_256_bits_exactly_and_too_wide():
    r = np.random.default_rng(4)
    n = 50_000
    exps = r.integers(0, 2 ** 32, size=(n // 4, 8), dtype=np.uint64).astype(np.uint32)
    exps[0] = 0xffffffff                                             # all 256 bits set: the largest key there is
    exps = np.ascontiguousarray(exps[r.integers(0, n // 4, size=n)])
    coef = r.standard_normal(n)
    c, e, st = run(W.Poly(coef, exps), 0.0)
    assert st.key_bits == 256 and st.key_bytes == 32 and len(st.digit_bits) == 32
    assert_parity(oracle.simplify(coef, exps), c, e)
    assert (e[-1] == 0xffffffff).all()
    too = np.full((10, 9), 0xffffffff, np.uint32)
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(np.ones(10)), dev(too))
    assert ei.value.status == B.ERR_KEY_TOO_WIDE
    with pytest.raises(B.PolylabError) as ei:                        # polylab_pack_keys exposes (hi, lo) pairs only
        B.pack_keys(dev(exps))
    assert ei.value.status == B.ERR_KEY_TOO_WIDE


def test_wide_products_fused_and_materialised():
    """mul_simplify with 160-bit keys (20 variables, sums up to 254): carries cross the 64-bit limbs of the key addition."""
    r = np.random.default_rng(21)
    a = W.Poly(r.standard_normal(700), r.integers(0, 128, size=(700, 20)).astype(np.uint8))
    b = W.Poly(r.standard_normal(90), r.integers(0, 128, size=(90, 20)).astype(np.uint8))
    a.exps[0:699:3] = a.exps[1:700:3]
    a.exps[0], b.exps[0] = 127, 127                                  # every field at its maximum in one product
    res = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, 0.0)
    for flags in (0, B.FLAG_NO_FUSED_PACK, B.FLAG_SAFE_RANK):
        c, e, st = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), 0.0, return_stats=True, flags=flags)
        assert st.key_bits == 160 and st.key_bytes == 32
        assert_parity(res, c.cpu().numpy(), e.cpu().numpy())
    # a small wide product: the one-block path
    c, e, st = B.mul_simplify(dev(a.coef[:40]), dev(a.exps[:40]), dev(b.coef[:40]), dev(b.exps[:40]), 0.0, return_stats=True)
    assert st.small_path == 1 and st.key_bytes == 32
    assert_parity(oracle.mul_simplify(a.coef[:40], a.exps[:40], b.coef[:40], b.exps[:40], 0.0), c.cpu().numpy(), e.cpu().numpy())


def test_wide_runs_tolerance_and_strides():
    p = pooled(100_000, 20, 50, seed=2, hi=1 << 12, dtype=np.uint16)   # 240 bits, runs of ~50 crossing tile boundaries
    res = oracle.simplify(p.coef, p.exps, 0.5)
    c, e, st = run(p, 0.5)
    assert st.key_bits == 240
    assert_parity(res, c, e)
    cm = dev(np.ascontiguousarray(p.exps.T)).T                         # column-major (MATLAB's pow, reading A13)
    c2, e2 = B.simplify(dev(p.coef), cm, 0.5)[:2]
    assert (e2.cpu().numpy() == e).all() and (c2.cpu().numpy() == c).all()
    n = 30_000                                                          # one run of equal wide keys spanning many tiles
    coef = np.random.default_rng(1).standard_normal(n)
    exps = np.tile(np.arange(1, 31, dtype=np.uint8) * 8, (n, 1))
    c, e, st = run(W.Poly(coef, exps), 0.0)
    assert len(c) == 1 and st.key_bytes == 32 and abs(c[0] - coef.sum()) <= 1e-12 * np.abs(coef).sum()


def test_wide_batched_matrix_product():
    r = np.random.default_rng(33)
    nv, nt = 30, 12

    def mat():
        c = r.standard_normal(4 * nt)
        e = r.integers(0, 100, size=(4 * nt, nv)).astype(np.uint8)
        return c, e, np.arange(5, dtype=np.int64) * nt
    A, Bm = mat(), mat()
    c, e, off, st = B.matmul_simplify(dev(A[0]), dev(A[1]), A[2], dev(Bm[0]), dev(Bm[1]), Bm[2], 2, 2, 2, 0.0, return_stats=True)
    c, e = c.cpu().numpy(), e.cpu().numpy()
    assert st.key_bytes == 32 and st.key_bits == 30 * 8 + 2
    for i in range(2):
        for j in range(2):
            cs, es = [], []
            for l in range(2):
                a0, a1, b0, b1 = A[2][i * 2 + l], A[2][i * 2 + l + 1], Bm[2][l * 2 + j], Bm[2][l * 2 + j + 1]
                pc, pe = oracle.expand(A[0][a0:a1], A[1][a0:a1], Bm[0][b0:b1], Bm[1][b0:b1])
                cs.append(pc)
                es.append(pe)
            q = i * 2 + j
            assert_parity(oracle.simplify(np.concatenate(cs), np.concatenate(es), 0.0), c[off[q]:off[q + 1]], e[off[q]:off[q + 1]])

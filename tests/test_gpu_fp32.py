"""-m gpu: single-precision coefficient STORAGE (opts->coef_type = POLYLAB_COEF_F32; the paper's
polylab_precision('set','single'), Table 10).  fp32 inputs are widened on their first
load, all arithmetic stays fp64, a result is rounded to fp32 once when stored.  Oracle: the same fp32 values converted
exactly to fp64, the oracle's sums s_m, expected output fl32(s_m); bound |gpu - s_m| <= 2^-24 |s_m| + 1e-12 A_m."""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import dev

pytestmark = pytest.mark.gpu


def check32(res, c, e, what=""):
    """Monomial set and order bit-exact (outside the exemption band), coefficients within the fp32 storage bound."""
    c = np.asarray(c.cpu().numpy() if isinstance(c, torch.Tensor) else c)
    e = np.asarray(e.cpu().numpy() if isinstance(e, torch.Tensor) else e)
    assert c.dtype == np.float32, what
    band = np.abs(np.abs(res.sum) - res.tol) <= 1e-12 * res.abs
    must = res.keep & ~band
    rows = {tuple(r): i for i, r in enumerate(res.rows.tolist())}
    got = [rows.get(tuple(r)) for r in e.tolist()]
    assert all(g is not None for g in got), what + ": a monomial that is not in the input"
    assert got == sorted(got) and len(set(got)) == len(got), what + ": not strictly ascending"
    gi = np.array(got, dtype=np.int64)
    present = np.zeros(len(res.sum), bool)
    present[gi] = True
    assert not (must & ~present).any(), what + ": a monomial is missing"
    assert not (present & ~res.keep & ~band).any(), what + ": a monomial should have been pruned"
    s, a = res.sum[gi], res.abs[gi]
    assert (np.abs(c.astype(np.float64) - s) <= 2.0 ** -24 * np.abs(s) + 1e-12 * a + 1e-45).all(), what + ": coefficient out of the fp32 bound"


def f32poly(p):
    return W.Poly(p.coef.astype(np.float32), p.exps)


@pytest.mark.parametrize("cfg,flags", [("c1", 0), ("c1", B.FLAG_NO_TABLE), ("c1small", 0), ("c3", 0), ("c3", B.FLAG_NO_TABLE),
                                       ("c5", 0), ("c5", B.FLAG_NO_BUCKET), ("c3u", 0), ("wide", 0)])
def test_simplify_fp32_on_every_path(cfg, flags):
    if cfg == "c1":
        p, tol = W.config1(100_000)
    elif cfg == "c1small":
        p, tol = W.config1(5000)
    elif cfg == "c3":
        p, tol = W.config3(400_000)
    elif cfg == "c5":
        p, tol = W.config5(2_000_000)
    elif cfg == "c3u":
        p, tol = W.config3u(200_000)
    else:
        r = np.random.default_rng(1)
        pool = r.integers(0, 256, size=(5000, 24), dtype=np.uint8)
        p, tol = W.Poly(r.standard_normal(60_000), np.ascontiguousarray(pool[r.integers(0, 5000, size=60_000)])), 0.0
    p = f32poly(p)
    res = oracle.simplify(p.coef.astype(np.float64), p.exps, tol)
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, flags=flags)
    check32(res, c, e, f"{cfg} flags {flags:#x}")
    if cfg == "c5":
        assert len(c) == p.nterms // 20 and st.prefix_passes == (2 if flags == 0 else 0)


def test_products_powers_batches_and_raw_expansion_in_fp32():
    a, b, tol = W.config2(600)
    a, b = f32poly(a), f32poly(b)
    res = oracle.mul_simplify(a.coef.astype(np.float64), a.exps, b.coef.astype(np.float64), b.exps, tol)
    for flags in (0, B.FLAG_NO_TABLE, B.FLAG_NO_TABLE | B.FLAG_NO_FUSED_PACK, B.FLAG_SAFE_RANK):
        c, e = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, flags=flags)
        check32(res, c, e, f"mul flags {flags:#x}")
    # the raw product: fp32 x fp32 is exact in fp64, so the stored value is the correctly rounded product
    rc, re_ = B.expand(dev(a.coef[:50]), dev(a.exps[:50]), dev(b.coef[:40]), dev(b.exps[:40]))
    oc, oe = oracle.expand(a.coef[:50].astype(np.float64), a.exps[:50], b.coef[:40].astype(np.float64), b.exps[:40])
    assert rc.dtype == torch.float32 and (re_.cpu().numpy() == oe).all()
    assert (rc.cpu().numpy() == oc.astype(np.float32)).all()
    # p^3 with packed fp64 intermediates and fp32 ends
    p = f32poly(W.config4()[0])
    c, e = B.pow_simplify(dev(p.coef), dev(p.exps), 3, 0.0, out_capacity=300_000)
    pc = p.coef.astype(np.float64)
    q = oracle.mul_simplify(pc, p.exps, pc, p.exps, 0.0)
    res3 = oracle.mul_simplify(*q.pruned, pc, p.exps.astype(np.uint32), 0.0)
    check32(res3, c, e, "pow")
    c, e = B.pow_simplify(dev(p.coef), dev(p.exps), 0)
    assert c.dtype == torch.float32 and c.cpu().tolist() == [1.0]
    # a 2x2 matrix product
    r = np.random.default_rng(3)
    nt = 30
    mk = lambda: (r.standard_normal(4 * nt).astype(np.float32), r.integers(0, 4, size=(4 * nt, 3)).astype(np.uint8), np.arange(5, dtype=np.int64) * nt)
    A, Bm = mk(), mk()
    c, e, off = B.matmul_simplify(dev(A[0]), dev(A[1]), A[2], dev(Bm[0]), dev(Bm[1]), Bm[2], 2, 2, 2, 0.0)
    c, e = c.cpu().numpy(), e.cpu().numpy()
    for i in range(2):
        for j in range(2):
            cs, es = zip(*[oracle.expand(A[0][A[2][i * 2 + l]:A[2][i * 2 + l + 1]].astype(np.float64), A[1][A[2][i * 2 + l]:A[2][i * 2 + l + 1]],
                                         Bm[0][Bm[2][l * 2 + j]:Bm[2][l * 2 + j + 1]].astype(np.float64), Bm[1][Bm[2][l * 2 + j]:Bm[2][l * 2 + j + 1]])
                           for l in range(2)])
            q = i * 2 + j
            check32(oracle.simplify(np.concatenate(cs), np.concatenate(es), 0.0), c[off[q]:off[q + 1]], e[off[q]:off[q + 1]], f"entry {q}")


def test_fp32_prune_uses_the_fp64_sum_and_mixed_dtypes_are_rejected():
    # 1 + 2^-30 - 1: the fp64 sum is 2^-30 (kept at tol = 0); summed in fp32 it would be 0
    coef = np.array([1.0, 2.0 ** -30, -1.0], np.float32)
    exps = np.array([[1], [1], [1]], np.uint8)
    for flags in (0, B.FLAG_DEBUG_FORCE_TABLE, B.FLAG_NO_SMALL):
        c, e = B.simplify(dev(coef), dev(exps), 0.0, flags=flags)
        assert e.cpu().tolist() == [[1]] and c.cpu().tolist() == [2.0 ** -30]
    with pytest.raises(B.PolylabError):
        B.mul_simplify(dev(coef), dev(exps), dev(coef.astype(np.float64)), dev(exps))
    # asynchronous call, fp32
    p = f32poly(W.config1(50_000)[0])
    oc = torch.empty(p.nterms, dtype=torch.float32, device="cuda")
    oe = torch.empty((p.nterms, 4), dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    status = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    B.simplify_async(dev(p.coef), dev(p.exps), 0.0, [3, 3, 3, 3], oc, oe, cnt, status)
    torch.cuda.synchronize()
    k = int(cnt.item())
    assert int(status.item()) == 0 and k == 256
    check32(oracle.simplify(p.coef.astype(np.float64), p.exps, 0.0), oc[:k], oe[:k], "async")


@pytest.mark.parametrize("seed", range(30))
def test_fuzz_fp32(seed):
    r = np.random.default_rng(77_000 + seed)
    dtype = [np.uint8, np.uint16][seed % 2]
    nvars = int(r.choice([1, 3, 8, 17, 33]))
    his = [int(r.choice([2, 4, 16, 200, 256])) for _ in range(nvars)]
    n = int(r.choice([1, 700, 4097, 8192, 8193, 40000, 200000]))
    dup = int(r.choice([1, 4, 50, 1000]))
    pool = np.stack([r.integers(0, h, size=max(1, n // dup)) for h in his], axis=1).astype(dtype)
    exps = np.ascontiguousarray(pool[r.integers(0, len(pool), size=n)])
    coef = r.standard_normal(n).astype(np.float32)
    tol = [0.0, 0.5][seed % 2]
    res = oracle.simplify(coef.astype(np.float64), exps, tol)
    for fl in (0, B.FLAG_NO_TABLE, B.FLAG_NO_TABLE | B.FLAG_NO_SMALL, B.FLAG_DEBUG_FORCE_TABLE | B.FLAG_DEBUG_FORCE_HASH,
               B.FLAG_DEBUG_FORCE_BUCKET, B.FLAG_SAFE_RANK):
        c, e = B.simplify(dev(coef), dev(exps), tol, flags=fl)
        check32(res, c, e, f"seed {seed} flags {fl:#x} n {n}")

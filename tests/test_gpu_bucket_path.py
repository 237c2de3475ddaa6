"""-m gpu: the bucket path of the CUDA library (csrc/finish.cu: partition on the most significant digits, finish every
bucket in shared memory, fused segmented sum / prune / unpack) against the CPU oracle under the same parity rule, its
self-checks and its fallbacks.  POLYLAB_FLAG_DEBUG_FORCE_BUCKET lets small inputs reach the path."""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import assert_parity, dev

pytestmark = pytest.mark.gpu

FORCE = B.FLAG_DEBUG_FORCE_BUCKET


def run(p, tol, flags=0, **kw):
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, flags=flags, **kw)
    torch.cuda.synchronize()
    return c.cpu().numpy(), e.cpu().numpy(), st


def pooled(n, nvars, dup, seed, hi=256, dtype=np.uint8):
    """n terms drawn from a pool of n/dup uniform monomials (config 5's structure, any width), coef N(0,1)."""
    r = np.random.default_rng(seed)
    pool = r.integers(0, hi, size=(n // dup, nvars)).astype(dtype)
    exps = pool[r.permutation(n) // dup]
    return W.Poly(r.standard_normal(n), np.ascontiguousarray(exps))


def test_config5_takes_the_bucket_path_by_default():
    """2e6 terms of config 5: 16 digits, 2 prefix passes, then the finish; same answer as the LSD path."""
    p, tol = W.config5(2_000_000)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = run(p, tol)
    assert st.prefix_passes == 2 and st.sort_passes == 2 and st.bucket_fallback == 0 and st.rank_fallback == 0
    assert st.distinct == 200_000 and st.survivors == 100_000 == len(c)
    assert_parity(res, c, e)
    c1, e1, st1 = run(p, tol, flags=B.FLAG_NO_BUCKET)
    assert st1.prefix_passes == 0 and st1.sort_passes == 16
    assert_parity(res, c1, e1)
    assert (e == e1).all()
    c2, e2, _ = run(p, tol)                                 # bit-reproducible run to run
    assert (c.view(np.uint64) == c2.view(np.uint64)).all() and (e == e2).all()


@pytest.mark.parametrize("n", [20, 10_000, 100_000, 300_000])
def test_forced_bucket_path_small_config5(n):
    p, tol = W.config5(n)
    c, e, st = run(p, tol, flags=FORCE)
    assert st.prefix_passes >= 1 and st.bucket_fallback == 0
    assert len(c) == n // 20
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


def test_fast_digit_list_too_short_is_detected_and_resorted():
    """With one fast digit (8 bits below the prefix) most tiles hold distinct keys that agree on it: the order check
    must catch them and the tile must re-sort on every low digit."""
    p, tol = W.config5(300_000)
    c, e, st = run(p, tol, flags=FORCE | (1 << B.FLAG_DEBUG_NFAST_SHIFT))
    assert st.prefix_passes == 1 and st.refinish_tiles > 0 and st.rank_fallback == 0
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)
    c3, e3, st3 = run(p, tol, flags=FORCE)                  # default list: no tile needs it here
    assert st3.refinish_tiles == 0
    assert (e == e3).all() and (c.view(np.uint64) == c3.view(np.uint64)).all()


def test_skewed_prefix_overflows_and_falls_back_to_lsd():
    """Config 3's leading variables are mostly zero: one bucket holds a large share of the terms, does not fit a
    tile, and the call must re-run on the LSD path with the same result."""
    p, tol = W.config3(300_000)
    c, e, st = run(p, tol, flags=FORCE)
    assert st.bucket_fallback == 1 and st.prefix_passes == 0 and st.sort_passes == 4
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


def test_skewed_prefix_is_rejected_by_the_histogram_precheck():
    """Default flags, 1.2e6 terms of config 3u (110-bit keys): the first prefix digit's histogram is far from flat, so
    the bucket path is dropped before any pass runs."""
    p, tol = W.config3u(1_200_000)
    c, e, st = run(p, tol)
    assert st.key_bits == 110 and st.bucket_fallback == 1 and st.prefix_passes == 0 and st.sort_passes == 14
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


def test_64_bit_keys_default_bucket_path():
    p = pooled(1_200_000, 8, 4, seed=11)
    c, e, st = run(p, 0.0)
    assert st.key_bytes == 8 and st.prefix_passes == 2 and st.bucket_fallback == 0
    assert len(c) == st.distinct
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


def test_72_bit_keys_prefix_digit_in_its_own_word():
    """9 variables of 8 bits: the top digit sits alone in the third 32-bit word of the key."""
    p = pooled(200_000, 9, 5, seed=12)
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.key_bits == 72 and st.key_bytes == 16 and st.prefix_passes == 1
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


@pytest.mark.parametrize("n", [1, 2, 33, 3000, 3584])
def test_forced_one_bucket_of_equal_keys(n):
    """All terms share one monomial: one bucket, one run, inside one finish tile."""
    r = np.random.default_rng(n)
    p = W.Poly(r.standard_normal(n), np.tile(np.array([[200, 3, 0, 77, 1, 2, 3, 4, 5]], np.uint8), (n, 1)))
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.prefix_passes >= 1 and st.bucket_fallback == 0 and len(c) == 1
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


def test_forced_one_bucket_too_long_falls_back():
    n = 20_000
    r = np.random.default_rng(5)
    exps = np.tile(np.array([[9, 9, 9, 9, 9]], np.uint8), (n, 1))
    exps[:, 4] = r.integers(0, 256, n)                      # same prefix, 256 monomials
    p = W.Poly(r.standard_normal(n), exps)
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.bucket_fallback == 1 and len(c) == 256
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


def test_forced_all_distinct_and_many_tiny_buckets():
    """Every term its own monomial, three prefix passes' worth of tiny buckets inside each tile (ordinal passes > 1)."""
    n = 100_003
    r = np.random.default_rng(7)
    exps = r.integers(0, 256, size=(n, 12)).astype(np.uint8)
    p = W.Poly(r.standard_normal(n), exps)
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.prefix_passes >= 1 and len(c) == len(np.unique(exps, axis=0))
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


def test_bucket_path_prune_capacity_and_p_minus_p():
    p, tol = W.config5(200_000)
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p.coef), dev(p.exps), tol, out_capacity=100, flags=FORCE)
    assert ei.value.status == B.ERR_OUTPUT_TOO_SMALL
    q = W.Poly(np.concatenate([p.coef, -p.coef]), np.concatenate([p.exps, p.exps]))
    c, e, st = run(q, 1e-12, flags=FORCE)
    assert st.prefix_passes >= 1 and len(c) == 0


def test_bucket_path_mul_simplify():
    """Product of two 1100-term polynomials over 8 variables with exponents up to 127: 1.21e6 products, 64-bit keys."""
    r = np.random.default_rng(21)
    a = W.Poly(r.standard_normal(1100), r.integers(0, 128, size=(1100, 8)).astype(np.uint8))
    b = W.Poly(r.standard_normal(1100), r.integers(0, 128, size=(1100, 8)).astype(np.uint8))
    c, e, st = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), 0.0, return_stats=True)
    assert st.prefix_passes >= 1 and st.bucket_fallback == 0
    assert_parity(oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, 0.0), c.cpu().numpy(), e.cpu().numpy())


# ------------------------------------------------------------------ S1 fused into the first radix pass

@pytest.mark.parametrize("case", ["u8x16_bytes", "u8x16_narrow", "u8x8", "u16x8", "u32x4", "u32x2", "u16x4"])
def test_fused_pack_matches_separate_pack(case):
    """Rows of 8 or 16 contiguous bytes are packed inside the first prefix pass; the result must be bit-identical to
    the run with S1 as its own kernel (POLYLAB_FLAG_NO_FUSED_PACK), and in parity with the oracle."""
    n = 120_000
    nvars, dtype, hi = {"u8x16_bytes": (16, np.uint8, 256), "u8x16_narrow": (16, np.uint8, 100), "u8x8": (8, np.uint8, 256),
                        "u16x8": (8, np.uint16, 5000), "u32x4": (4, np.uint32, 70000), "u32x2": (2, np.uint32, 1 << 20),
                        "u16x4": (4, np.uint16, 40000)}[case]
    p = pooled(n, nvars, 4, seed=31 + nvars, hi=hi, dtype=dtype)
    c, e, st = run(p, 0.0, flags=FORCE)
    c0, e0, st0 = run(p, 0.0, flags=FORCE | B.FLAG_NO_FUSED_PACK)
    assert st.prefix_passes >= 1 and st0.prefix_passes == st.prefix_passes
    assert st.kernel_launches == st0.kernel_launches          # row histogram instead of the pack kernel
    assert (e == e0).all() and (c.view(np.uint64) == c0.view(np.uint64)).all()
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


def test_fused_pack_checks_caller_bounds():
    p = pooled(50_000, 16, 4, seed=41, hi=200)
    with pytest.raises(B.PolylabError) as ei:
        B.simplify(dev(p.coef), dev(p.exps), 0.0, max_exp=[150] * 16, flags=FORCE)
    assert ei.value.status == B.ERR_EXPONENT_RANGE
    c, e, st = B.simplify(dev(p.coef), dev(p.exps), 0.0, max_exp=[255] * 16, flags=FORCE, return_stats=True)
    assert st.prefix_passes >= 1
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c.cpu().numpy(), e.cpu().numpy())


def test_unstable_prefix_passes_are_detected_on_the_bucket_path():
    """POLYLAB_FLAG_DEBUG_UNSTABLE breaks the stability of the radix passes; with two prefix passes the array is then not
    sorted by prefix, the finish kernel's prefix-order checks (inside a tile and at every tile start) must see it and the
    call must re-run on the LSD path with ballot ranking."""
    p, tol = W.config5(2_000_000)
    c, e, st = run(p, tol, flags=B.FLAG_DEBUG_UNSTABLE)
    assert st.rank_fallback == 1 and st.prefix_passes == 0 and st.sort_passes == 16
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


@pytest.mark.parametrize("seed", range(40))
def test_randomised_shapes_both_paths(seed):
    """Random variable counts, dtypes, exponent ranges, duplication and sizes: the forced bucket path and the LSD path
    must both be in parity with the oracle and agree on the monomial set (a poor man's fuzzer; compute-sanitizer is
    not available on the GPU pool)."""
    r = np.random.default_rng(1000 + seed)
    dtype = [np.uint8, np.uint16, np.uint32][int(r.integers(0, 3))]
    nvars = int(r.integers(1, 17))
    his = r.choice([1, 2, 4, 16, 200, 256, 1000, 60000][: {np.uint8: 6, np.uint16: 8, np.uint32: 8}[dtype]], size=nvars)
    while sum(int(h - 1).bit_length() for h in his) > 128:          # keep the key within 128 bits
        his[int(r.integers(0, nvars))] = 2
    n = int(r.choice([1, 7, 300, 4607, 4609, 20_000, 60_001]))
    dup = int(r.choice([1, 2, 5, 50]))
    pool = np.stack([r.integers(0, h, size=max(1, n // dup)) for h in his], axis=1).astype(dtype)
    exps = np.ascontiguousarray(pool[r.integers(0, len(pool), size=n)])
    coef = r.standard_normal(n)
    if seed % 4 == 0:
        coef[: n // 2] = -coef[n - n // 2:][::-1]                    # some cancellation
    tol = [0.0, 1e-14, 0.5][seed % 3]
    p = W.Poly(coef, exps)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = run(p, tol, flags=FORCE)
    assert_parity(res, c, e)
    c0, e0, st0 = run(p, tol, flags=B.FLAG_NO_BUCKET | B.FLAG_NO_TABLE)
    assert st0.prefix_passes == 0 and st0.table_path == 0
    assert_parity(res, c0, e0)
    if tol == 0.0:
        assert (e == e0).all()
    if sum(int(h - 1).bit_length() for h in his) <= 63:             # the table path (table.cu), dense or hash, and hash alone
        for fl in (B.FLAG_DEBUG_FORCE_TABLE, B.FLAG_DEBUG_FORCE_TABLE | B.FLAG_DEBUG_FORCE_HASH):
            c1, e1, st1 = run(p, tol, flags=fl)
            assert_parity(res, c1, e1)
            assert st1.table_path in (1, 2) or st1.table_fallback == 1 or st1.key_bits == 0


# ------------------------------------------------------------------ S0 on a sample of the rows

def test_sampled_bounds_are_verified_and_retried():
    """>= 2^22 terms: S0 reads a sample of the rows and S1's range check verifies the rest.  An exponent the sample misses
    (one row of 200 among values below 16) must be caught and the call re-run with full bounds -- same result as
    POLYLAB_FLAG_EXACT_BOUNDS."""
    n = (1 << 22) + 12_344
    p = pooled(n, 8, 8, seed=51, hi=16)
    c, e, st = run(p, 0.0)
    assert st.bounds_sampled == 1 and st.bounds_retry == 0 and st.key_bits == 32
    res = oracle.simplify(p.coef, p.exps, 0.0)
    assert_parity(res, c, e)
    p.exps[1000, 3] = 200                                   # rows 512..3500 of every stride are not sampled
    res = oracle.simplify(p.coef, p.exps, 0.0)
    c, e, st = run(p, 0.0)
    assert st.bounds_retry == 1 and st.bounds_sampled == 0 and st.key_bits == 36
    assert_parity(res, c, e)
    c1, e1, st1 = run(p, 0.0, flags=B.FLAG_EXACT_BOUNDS)
    assert st1.bounds_retry == 0 and st1.bounds_sampled == 0
    assert (e == e1).all() and (c.view(np.uint64) == c1.view(np.uint64)).all()


def test_out_of_range_exponents_on_the_fused_path_are_reported_not_scattered():
    """Caller bounds far too small (4-bit fields, exponents up to 199): the fused pass clamps what it reports, so its
    scatter still agrees with the digit histogram built from the rows, and the call returns the range error."""
    p = pooled(300_000, 16, 4, seed=61, hi=200)
    for _ in range(3):
        with pytest.raises(B.PolylabError) as ei:
            B.simplify(dev(p.coef), dev(p.exps), 0.0, max_exp=[15] * 16, flags=FORCE)
        assert ei.value.status == B.ERR_EXPONENT_RANGE
    c, e, st = run(p, 0.0, flags=FORCE)                     # the library is still healthy afterwards
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


def test_sampled_bounds_retry_on_the_bucket_path_with_fused_pack():
    n = (1 << 22) + 8_000
    p = pooled(n, 16, 8, seed=52, hi=16)
    p.exps[2000, 5] = 200                                   # not in the sample
    c, e, st = run(p, 0.0)
    assert st.bounds_retry == 1 and st.key_bits == 68 and st.prefix_passes == 2
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)


# ------------------------------------------------------------------ asynchronous calls on the fast path

def _async(p, tol, flags=0, with_status=True):
    n = p.nterms
    oc = torch.empty(n, dtype=torch.float64, device="cuda")
    oe = torch.empty((n, p.nvars), dtype=torch.uint8, device="cuda")
    cnt = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    status = torch.full((1,), -1, dtype=torch.int32, device="cuda") if with_status else None
    st = B.simplify_async(dev(p.coef), dev(p.exps), tol, [255] * p.nvars, oc, oe, cnt, status, flags=flags)
    torch.cuda.synchronize()
    k = int(cnt.item())
    return oc[:k].cpu().numpy(), oe[:k].cpu().numpy(), (int(status.item()) if with_status else None), st


def test_async_call_takes_the_bucket_path():
    """POLYLAB_FLAG_DEVICE_COUNT with a status word: no host synchronisation, yet atomic ranking, fused pack and the bucket
    path -- the self-checks report through status_device (POLYLAB_ERR_RETRY) instead of a read-back."""
    p, tol = W.config5(2_000_000)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, status, st = _async(p, tol)
    assert status == B.OK and st.prefix_passes == 2 and len(c) == 100_000
    assert_parity(res, c, e)
    c0, e0, _ = run(p, tol)                                       # the synchronous call: same kernels, same bits
    assert (e0 == e).all() and (c0.view(np.uint64) == c.view(np.uint64)).all()
    # an unstable ranking (test hook) is reported, not hidden: status RETRY, count 0
    c, e, status, st = _async(p, tol, flags=B.FLAG_DEBUG_UNSTABLE)
    assert status == B.ERR_RETRY and len(c) == 0
    # the retry the header prescribes
    c, e, status, st = _async(p, tol, flags=B.FLAG_SAFE_RANK | B.FLAG_NO_BUCKET)
    assert status == B.OK and st.prefix_passes == 0
    assert_parity(res, c, e)
    # without a status word the call must not depend on a check nobody could read: ballot ranking, LSD passes
    c, e, status, st = _async(p, tol, with_status=False)
    assert st.prefix_passes == 0 and st.sort_passes == 16
    assert_parity(res, c, e)
    # a skewed prefix (one huge bucket): tile_bounds_kernel raises overflow -> RETRY
    q = pooled(300_000, 16, 10, seed=3)
    q.exps[:, :2] = 7
    c, e, status, st = _async(q, 0.0, flags=FORCE)
    assert status == B.ERR_RETRY and len(c) == 0
    c, e, status, st = _async(q, 0.0, flags=B.FLAG_SAFE_RANK | B.FLAG_NO_BUCKET)
    assert status == B.OK
    assert_parity(oracle.simplify(q.coef, q.exps, 0.0), c, e)


# ------------------------------------------------------------------ slack bins from a sampled histogram

def test_slack_bins_match_the_exact_histogram_bit_for_bit():
    """>= 2^22 terms, fused pack, two prefix passes: the first pass's bins are laid out with slack from a sampled histogram and
    the second pass reads through the holes -- same records in the same order as with the exact sweep, so identical bits."""
    n = (1 << 22) + 16
    p, tol = W.config5(n)
    c, e, st = run(p, tol)
    assert st.hist_sampled == 1 and st.hist_retry == 0 and st.prefix_passes == 2
    c1, e1, st1 = run(p, tol, flags=B.FLAG_EXACT_HIST)
    assert st1.hist_sampled == 0 and st1.prefix_passes == 2
    assert (e == e1).all() and (c.view(np.uint64) == c1.view(np.uint64)).all()
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)
    # 64-bit keys (rows of 8 bytes), non-uniform but smooth first digit
    r = np.random.default_rng(5)
    m = 6_000_000
    pool = r.integers(0, 256, size=(m // 6, 8)).astype(np.uint8)
    pool[:, 1] = (r.integers(0, 256, size=m // 6) * r.integers(0, 256, size=m // 6) // 256).astype(np.uint8)   # triangular-ish
    q = W.Poly(r.standard_normal(m), np.ascontiguousarray(pool[r.integers(0, m // 6, size=m)]))
    c, e, st = run(q, 0.0, flags=B.FLAG_NO_TABLE)
    assert st.key_bytes == 8
    assert_parity(oracle.simplify(q.coef, q.exps, 0.0), c, e)
    if st.hist_sampled:
        c1, e1, _ = run(q, 0.0, flags=B.FLAG_NO_TABLE | B.FLAG_EXACT_HIST)
        assert (e == e1).all() and (c.view(np.uint64) == c1.view(np.uint64)).all()


def test_slack_bin_overrun_is_detected_and_the_call_reruns():
    """An input whose sampled segments are NOT representative: the rows the sample never reads (segments of 2048 rows every
    16,891) all share one value of the first prefix digit, so that bin overruns its capacity -> the pass raises slack_overflow,
    the call re-runs with the exact sweep (stats->hist_retry) and still agrees with the oracle."""
    n = 20_000_020
    p, tol = W.config5(n)
    exps = p.exps.copy()
    stride = n // (148 * 8)
    pos = np.arange(n) % stride
    exps[pos >= 2048, 1] = 7                                   # the second variable is the first prefix digit (T = 16: digits of variables 0, 1)
    q = W.Poly(p.coef, exps)
    c, e, st = run(q, tol)
    assert st.hist_retry == 1 and st.hist_sampled == 0
    assert_parity(oracle.simplify(q.coef, q.exps, tol), c, e)


def test_async_call_uses_slack_bins_with_capacities_computed_on_the_device():
    """POLYLAB_FLAG_DEVICE_COUNT at >= 2^22 terms: the sampled histogram never reaches the host (slack_caps_kernel sizes the
    bins); same bits as the synchronous call.  An unrepresentative sample (the input of the test above) cannot re-run
    without a read-back: status POLYLAB_ERR_RETRY, count 0, and the prescribed retry gives the oracle's result."""
    n = (1 << 22) + 16
    p, tol = W.config5(n)
    c, e, status, st = _async(p, tol)
    assert status == B.OK and st.prefix_passes == 2 and st.hist_sampled == 1 and len(c) == n // 20
    c0, e0, st0 = run(p, tol)
    assert st0.hist_sampled == 1
    assert (e0 == e).all() and (c0.view(np.uint64) == c.view(np.uint64)).all()
    exps = p.exps.copy()
    stride = n // (148 * 8)
    exps[(np.arange(n) % stride) >= 2048, 1] = 7
    q = W.Poly(p.coef, exps)
    c, e, status, st = _async(q, tol)
    assert status == B.ERR_RETRY and len(c) == 0
    c, e, status, st = _async(q, tol, flags=B.FLAG_SAFE_RANK | B.FLAG_NO_BUCKET)
    assert status == B.OK
    assert_parity(oracle.simplify(q.coef, q.exps, tol), c, e)


# ---------------------------------------------------------------------------------- group kernel (finish.cu, round 2)

def _bits(c, e):
    return c.view(np.uint64).copy(), e.copy()


def test_group_finish_is_taken_and_matches_the_sorting_finish_bit_for_bit():
    """Config 5's structure (ten records per monomial): the tiles are finished by grouping like terms in the shared-memory hash
    table; the sorting kernel alone (POLYLAB_FLAG_NO_GROUP_FINISH) and the group kernel handing every tile on give the same bits."""
    p, tol = W.config5(2_000_000)
    res = oracle.simplify(p.coef, p.exps, tol)
    c, e, st = run(p, tol)
    assert st.prefix_passes == 2 and st.bucket_fallback == 0 and st.rank_fallback == 0
    assert st.grouped_tiles > 0
    assert_parity(res, c, e)
    c0, e0, st0 = run(p, tol, flags=B.FLAG_NO_GROUP_FINISH)
    assert st0.grouped_tiles == 0 and st0.prefix_passes == 2
    c1, e1, st1 = run(p, tol, flags=B.FLAG_DEBUG_GROUP_HANDS_ON)
    assert st1.grouped_tiles == 0 and st1.prefix_passes == 2
    assert st.distinct == st0.distinct == st1.distinct and st.survivors == st0.survivors == st1.survivors
    for cc, ee in ((c0, e0), (c1, e1)):
        assert (e == ee).all() and (c.view(np.uint64) == cc.view(np.uint64)).all()
    c2, e2, st2 = run(p, tol)                               # bit-reproducible run to run
    assert (c.view(np.uint64) == c2.view(np.uint64)).all() and (e == e2).all()


@pytest.mark.parametrize("n,nvars,dup,seed", [(300_000, 9, 10, 1), (300_000, 16, 3, 2), (1_200_000, 8, 4, 3), (1_200_000, 12, 40, 4),
                                              (150_003, 5, 7, 5), (2_500_000, 16, 1, 6), (600_000, 10, 40, 7)])
def test_group_finish_shapes(n, nvars, dup, seed):
    """One- and two-word keys, one bucket per tile and dozens of buckets per tile (the composite word's prefix difference),
    heavy and no duplication (tiles with more than 768 distinct keys are handed on): oracle parity and the same bits as the
    sorting kernel."""
    p = pooled(n, nvars, dup, seed)
    res = oracle.simplify(p.coef, p.exps, 0.0)
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.prefix_passes >= 1 and st.bucket_fallback == 0
    assert_parity(res, c, e)
    c0, e0, st0 = run(p, 0.0, flags=FORCE | B.FLAG_NO_GROUP_FINISH)
    assert st0.grouped_tiles == 0 and st0.prefix_passes == st.prefix_passes
    assert (e == e0).all() and (c.view(np.uint64) == c0.view(np.uint64)).all()
    if dup >= 3 and n // dup < 100_000:
        assert st.grouped_tiles > 0


def test_group_finish_cancelling_terms_and_tolerance():
    """p - p through the group kernel: every run sums to exactly zero and is pruned at tol = 0; with a tolerance the parity rule's
    exemption band applies as everywhere."""
    r = np.random.default_rng(21)
    base = pooled(400_000, 16, 8, seed=22)
    p = W.Poly(np.concatenate([base.coef, -base.coef]), np.concatenate([base.exps, base.exps]))
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.grouped_tiles > 0
    res = oracle.simplify(p.coef, p.exps, 0.0)
    assert_parity(res, c, e)
    q = W.Poly(r.standard_normal(len(p.coef)), p.exps)
    c, e, st = run(q, 1e-3, flags=FORCE)
    assert st.grouped_tiles > 0
    assert_parity(oracle.simplify(q.coef, q.exps, 1e-3), c, e)


def test_group_finish_short_fast_digit_list_hands_tiles_on():
    """With 8 sort bits below the prefix the group kernel's sort of the distinct keys fails its order check: such tiles go
    through the sorting kernel, which re-sorts them on every digit."""
    p, tol = W.config5(300_000)
    c, e, st = run(p, tol, flags=FORCE | (1 << B.FLAG_DEBUG_NFAST_SHIFT))
    assert st.refinish_tiles > 0
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c, e)


def test_group_finish_crowded_leading_digit_hands_tiles_on():
    """Variables 1..3 take one value each, so every key of a bucket shares the ten bits below the prefix and all of a tile's
    distinct keys fall into one leading-digit bin: more than 16 of them, the group kernel hands the tile on and the sorting
    kernel finishes it.  Same answer, no grouped tile."""
    r = np.random.default_rng(31)
    n, dup = 400_000, 8
    pool = r.integers(0, 256, size=(n // dup, 9)).astype(np.uint8)
    pool[:, 1] = 255                                          # full-width fields (the layout is sized from the maxima) ...
    pool[:, 2] = 255
    pool[:, 3] = 255                                          # ... that never vary: 24 constant bits right below the first digit
    exps = np.ascontiguousarray(pool[r.permutation(n) // dup])
    p = W.Poly(r.standard_normal(n), exps)
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.prefix_passes == 1 and st.bucket_fallback == 0 and st.grouped_tiles == 0
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)
    c0, e0, _ = run(p, 0.0, flags=FORCE | B.FLAG_NO_GROUP_FINISH)
    assert (e == e0).all() and (c.view(np.uint64) == c0.view(np.uint64)).all()


def test_group_finish_mixed_tiles():
    """Half of the buckets hold few distinct monomials (grouped), the other half only distinct ones (more than 768 per tile:
    handed on, but never so many that the give-up rule fires): both kernels contribute to one output."""
    r = np.random.default_rng(32)
    nd, nu = 600_000, 600_000
    pd = r.integers(0, 256, size=(nd // 20, 8)).astype(np.uint8)
    pd[:, 0] &= 0x7f                                          # duplicated monomials under the low half of the first digit
    ed = pd[r.permutation(nd) // 20]
    eu = r.integers(0, 256, size=(nu, 8)).astype(np.uint8)
    eu[:, 0] |= 0x80                                          # distinct ones under the high half
    exps = np.ascontiguousarray(np.concatenate([ed, eu])[r.permutation(nd + nu)])
    p = W.Poly(r.standard_normal(nd + nu), exps)
    c, e, st = run(p, 0.0, flags=FORCE)
    assert st.prefix_passes >= 1 and st.bucket_fallback == 0
    assert 0 < st.grouped_tiles
    res = oracle.simplify(p.coef, p.exps, 0.0)
    assert_parity(res, c, e)
    c0, e0, st0 = run(p, 0.0, flags=FORCE | B.FLAG_NO_GROUP_FINISH)
    assert st0.grouped_tiles == 0 and (e == e0).all() and (c.view(np.uint64) == c0.view(np.uint64)).all()


def test_group_finish_without_like_terms_gives_up_and_matches():
    """2.4e6 distinct monomials: every tile holds more than 768 distinct keys; after the first tiles the group kernel stops
    trying (the give-up rule), the sorting kernel finishes everything."""
    p = pooled(2_400_000, 8, 1, seed=33)
    c, e, st = run(p, 0.0)
    assert st.prefix_passes == 2 and st.bucket_fallback == 0 and st.grouped_tiles == 0
    assert len(c) == st.distinct
    assert_parity(oracle.simplify(p.coef, p.exps, 0.0), c, e)

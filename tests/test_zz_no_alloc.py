"""-m gpu, collected last: polylab_simplify_static -- the entry point that allocates nothing (its scratch memory is a static
device array inside the library, include/polylab.h) -- against the existing path (polylab_simplify with a caller workspace)
and the CPU oracle, on calls in a row that share the array.  Same kernels, same order: the bits must agree; the parity rule
(1e-12 * A_m, oracle/parity.py) is checked as well."""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2604_06575_b200 import binding as B
from paper_2604_06575_b200 import workloads as W
from gpu_util import assert_parity, dev

pytestmark = pytest.mark.gpu


def _both(p, tol, **kw):
    c1, e1, st1 = B.simplify_static(dev(p.coef), dev(p.exps), tol, return_stats=True, **kw)
    c1, e1 = c1.cpu().numpy(), e1.cpu().numpy()
    c0, e0, st0 = B.simplify(dev(p.coef), dev(p.exps), tol, return_stats=True, **kw)
    c0, e0 = c0.cpu().numpy(), e0.cpu().numpy()
    return (c1, e1, st1), (c0, e0, st0)


def _agree(p, tol, **kw):
    (c1, e1, st1), (c0, e0, st0) = _both(p, tol, **kw)
    assert (st1.table_path, st1.small_path, st1.sort_passes) == (st0.table_path, st0.small_path, st0.sort_passes)
    assert e1.shape == e0.shape and (e1 == e0).all()
    A = max(float(np.abs(p.coef).sum()), 1e-300)
    assert np.all(np.abs(c1 - c0) <= 1e-12 * A)
    assert (c1.view(np.uint64) == c0.view(np.uint64)).all()          # the same kernels in the same order
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c1, e1)
    return st1


def test_static_workspace_matches_the_workspace_path_on_calls_in_a_row():
    # 1. the largest input the static array takes: config 1's recipe, dense table path
    p, tol = W.config1(B.STATIC_MAX_TERMS)
    st = _agree(p, tol)
    assert st.table_path == 1
    # 2. right after it, a SMALLER input on another path (one-block sort): the array still holds call 1's control block,
    #    table and tile states
    q, tol = W.config5(4000)                  # (the one-block path takes at most 4096 pairs with 128-bit keys)
    st = _agree(q, tol)
    assert st.small_path == 1 and st.key_bytes == 16
    # 3. radix passes over wide keys (table and one-block paths switched off), then the first input again
    r, tol = W.config5(50_000)
    st = _agree(r, tol, flags=B.FLAG_NO_TABLE)
    assert st.sort_passes == 16 and st.table_path == 0
    _agree(p, 0.0)
    # 4. the same call twice: identical bits
    a = B.simplify_static(dev(r.coef), dev(r.exps), tol)
    b = B.simplify_static(dev(r.coef), dev(r.exps), tol)
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])


def test_static_workspace_allocates_nothing_and_rejects_what_does_not_fit():
    p, tol = W.config3(40_000)
    coef, exps = dev(p.coef), dev(p.exps)
    out = (torch.empty(p.nterms, dtype=torch.float64, device="cuda"), torch.empty((p.nterms, p.nvars), dtype=torch.uint8, device="cuda"))
    B.simplify_static(coef, exps, tol, out=out)                     # first call on this device: the symbol lookup
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        c, e = B.simplify_static(coef, exps, tol, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                    # the driver handed out no device memory
    assert_parity(oracle.simplify(p.coef, p.exps, tol), c.cpu().numpy(), e.cpu().numpy())
    # one term more than the stated maximum: a clear error, nothing launched
    big, _ = W.config1(B.STATIC_MAX_TERMS + 1)
    with pytest.raises(B.PolylabError) as ei:
        B.simplify_static(dev(big.coef), dev(big.exps), 0.0)
    assert ei.value.status == B.ERR_WORKSPACE_TOO_SMALL
    with pytest.raises(B.PolylabError) as ei:                        # stage events would have to be created
        B.simplify_static(coef, exps, tol, flags=B.FLAG_TIMING)
    assert ei.value.status == B.ERR_INVALID_ARGUMENT
    # empty input
    c, e = B.simplify_static(coef[:0], exps[:0], 0.0)
    assert len(c) == 0

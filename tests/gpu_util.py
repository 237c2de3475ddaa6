"""Helpers shared by the -m gpu tests: run the CUDA path through the binding, the oracle on the same
seeded inputs, and apply the parity rule."""
import numpy as np
import torch

from oracle import oracle, parity
from paper_2604_06575_b200 import binding as B


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_simplify(coef, exps, tol=0.0, **kw):
    c, e = B.simplify(dev(coef), dev(exps), tol, **kw)[:2]
    torch.cuda.synchronize()
    return c.cpu().numpy(), e.cpu().numpy()


def gpu_mul(a, b, tol=0.0, **kw):
    c, e = B.mul_simplify(dev(a.coef), dev(a.exps), dev(b.coef), dev(b.exps), tol, **kw)[:2]
    torch.cuda.synchronize()
    return c.cpu().numpy(), e.cpu().numpy()


def assert_parity(res, c, e, **kw):
    rep = parity.check(res, c, e, **kw)
    assert rep.ok, str(rep)
    return rep


def check_simplify(coef, exps, tol=0.0, **kw):
    c, e = gpu_simplify(coef, exps, tol, **kw)
    res = oracle.simplify(coef, exps, tol)
    return assert_parity(res, c, e), (c, e), res


def check_mul(a, b, tol=0.0, **kw):
    c, e = gpu_mul(a, b, tol, **kw)
    res = oracle.mul_simplify(a.coef, a.exps, b.coef, b.exps, tol)
    return assert_parity(res, c, e), (c, e), res

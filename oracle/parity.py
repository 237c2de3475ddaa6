"""Parity rule between a simplified polynomial and the oracle's result.

TEST INFRASTRUCTURE (see oracle/oracle.py).  The rule is BASELINE.json's
north_star, restated (SURVEY.md 8(c) "Parity rule"):

  oracle: for every distinct monomial m of the input, s_m (merged coefficient)
  and A_m (sum of |contributing coefficients|); beta_m = 1e-12 * A_m.
  (1) m is EXEMPT from the set check iff | |s_m| - tol | <= beta_m;
  (2) otherwise m must be present in the candidate iff |s_m| > tol;
  (3) every candidate term is some m of the input (bit-exact exponents) and its
      coefficient g_m satisfies |g_m - s_m| <= beta_m;
  (4) the candidate's monomials are strictly ascending in lexicographic order,
      variable 0 most significant (reading A1).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

REL_TOL = 1e-12     # north_star: |gpu - oracle| <= 1e-12 * sum |contributing coefficients|


def _lexkey(rows: np.ndarray) -> np.ndarray:
    """Rows -> fixed-length byte strings whose byte order is the lexicographic row order."""
    rows = np.ascontiguousarray(rows)
    if rows.ndim != 2:
        raise ValueError("rows must be 2-D")
    n, nvars = rows.shape
    be = np.ascontiguousarray(rows.astype(">u4"))
    return be.view(f"S{4 * nvars}").reshape(n)


@dataclass
class ParityReport:
    ok: bool
    n_oracle_distinct: int
    n_expected: int          # oracle survivors
    n_candidate: int
    matched: int
    exempt: int
    max_rel_dev: float       # max |g - s| / A_m over matched terms with A_m > 0
    errors: list = field(default_factory=list)

    def __str__(self):
        head = (f"parity {'OK' if self.ok else 'FAIL'}: candidate {self.n_candidate} terms, oracle "
                f"{self.n_expected} survivors of {self.n_oracle_distinct} distinct; matched {self.matched}, "
                f"exempt {self.exempt}, max |g-s|/A = {self.max_rel_dev:.3e}")
        return head + "".join(f"\n  - {e}" for e in self.errors[:10])


def check(oracle_result, cand_coef, cand_rows, tol=None, rel=REL_TOL, subset_of_oracle=False) -> ParityReport:
    """Apply rules (1)-(4).  `oracle_result` is an oracle.OracleResult (unpruned list).

    subset_of_oracle=True skips rule (2)'s "must be present" half: the candidate
    is then a sample of the output (used for full-size sampled checks).
    """
    tol = oracle_result.tol if tol is None else float(tol)
    g = np.asarray(cand_coef, dtype=np.float64).reshape(-1)
    rows = np.asarray(cand_rows)
    if rows.ndim != 2:
        rows = rows.reshape(g.shape[0], -1)
    errors = []
    orows, s, a = oracle_result.rows, oracle_result.sum, oracle_result.abs
    nvars = orows.shape[1] if orows.size else (rows.shape[1] if rows.size else 0)
    if g.shape[0] != rows.shape[0]:
        errors.append(f"coef has {g.shape[0]} entries but rows has {rows.shape[0]}")
        return ParityReport(False, len(s), int(oracle_result.keep.sum()), int(g.shape[0]), 0, 0, float("nan"), errors)
    if rows.size and rows.shape[1] != nvars:
        errors.append(f"candidate has {rows.shape[1]} variables, oracle {nvars}")
        return ParityReport(False, len(s), int(oracle_result.keep.sum()), int(g.shape[0]), 0, 0, float("nan"), errors)

    beta = rel * a
    exempt = np.abs(np.abs(s) - tol) <= beta
    must = (np.abs(s) > tol) & ~exempt
    mustnot = ~(np.abs(s) > tol) & ~exempt

    ck = _lexkey(rows.astype(np.uint32)) if rows.size else np.zeros(0, "S4")
    ok_ = _lexkey(orows) if orows.size else np.zeros(0, "S4")

    # (4) strictly ascending canonical order
    if ck.shape[0] > 1:
        bad = np.nonzero(~(ck[1:] > ck[:-1]))[0]
        if bad.size:
            errors.append(f"candidate not strictly ascending at {bad.size} places, first at index {int(bad[0])}: "
                          f"{rows[bad[0]].tolist()} then {rows[bad[0] + 1].tolist()}")

    # (3) every candidate term is a monomial of the input, coefficient within beta_m
    present = np.zeros(len(s), dtype=bool)
    matched = 0
    max_rel = 0.0
    if ck.shape[0]:
        if ok_.shape[0] == 0:
            errors.append("candidate has terms but the input has no monomials")
        else:
            pos = np.searchsorted(ok_, ck)
            pos_c = np.minimum(pos, ok_.shape[0] - 1)
            found = ok_[pos_c] == ck
            if not found.all():
                i = int(np.nonzero(~found)[0][0])
                errors.append(f"{int((~found).sum())} candidate monomials do not occur in the input, e.g. "
                              f"{rows[i].tolist()} (coef {g[i]!r})")
            idx = pos_c[found]
            present[idx] = True
            dev = np.abs(g[found] - s[idx])
            bad = ~(dev <= beta[idx])          # NaN-safe: NaN fails
            matched = int(found.sum() - bad.sum())
            if bad.any():
                j = int(np.nonzero(bad)[0][0])
                errors.append(f"{int(bad.sum())} coefficients out of tolerance, e.g. monomial "
                              f"{orows[idx[j]].tolist()}: got {g[found][j]!r}, oracle {s[idx[j]]!r}, "
                              f"A_m {a[idx[j]]!r}")
            nz = a[idx] > 0
            if nz.any():
                max_rel = float(np.max(dev[nz] / a[idx][nz]))

    # (2) non-exempt monomials: present iff |s_m| > tol
    if not subset_of_oracle:
        missing = must & ~present
        if missing.any():
            j = int(np.nonzero(missing)[0][0])
            errors.append(f"{int(missing.sum())} monomials missing, e.g. {orows[j].tolist()} with s={s[j]!r}")
    extra = mustnot & present
    if extra.any():
        j = int(np.nonzero(extra)[0][0])
        errors.append(f"{int(extra.sum())} monomials should have been pruned, e.g. {orows[j].tolist()} "
                      f"with s={s[j]!r}, tol={tol!r}")

    return ParityReport(not errors, len(s), int(oracle_result.keep.sum()), int(g.shape[0]), matched,
                        int(exempt.sum()), max_rel, errors)

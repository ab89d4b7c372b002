"""The parity criterion GPU-vs-oracle, written out once ("Tolerance").

north_star rule: |d| <= 1e-12 |ref|, or |d| <= 1e-15 where |ref| < 1e-3.
Conditioning clause: an output whose weighted stencil magnitude S dwarfs |ref| (a sign change
of xf inside the cell) carries rounding noise ~eps*S in ANY fp64 evaluation order, the oracle's
included; such an output passes if |d| <= 1e-12 * S, S from the oracle's scale helper.
The count of outputs that needed the clause is reported and bounded.
"""
import numpy as np

REL = 1e-12
ABS_SMALL = 1e-15
SMALL = 1e-3
EPS_EQ1 = 1e-16  # PAPER.md:87-91, eq. 1


def eq1_rel_diff(got, ref):
    """r = |a - b| / (|b| + eps), eq. 1 of the paper."""
    return np.abs(got - ref) / (np.abs(ref) + EPS_EQ1)


def check_parity(got, ref, scale=None, max_clause_frac=2e-3, what="", clause_rel=REL):
    """Assert parity; returns a dict of statistics.

    ``clause_rel`` widens the conditioning clause only (never the north_star rule) for grids whose
    knots are much denser than the paper's: a last-bit difference in a coordinate logarithm moves
    t by ulp(u)/dU, so the clause scales with |u|/dU; the caller derives the factor."""
    got, ref = np.asarray(got), np.asarray(ref)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    nan_g, nan_r = np.isnan(got), np.isnan(ref)
    assert np.array_equal(nan_g, nan_r), f"{what}: NaN pattern differs"
    ok = ~nan_r
    d = np.abs(got[ok] - ref[ok])
    r = np.abs(ref[ok])
    rule = np.where(r < SMALL, d <= ABS_SMALL, d <= REL * r)
    n_clause = int((~rule).sum())
    stats = {"n": int(ok.sum()), "max_eq1": float(eq1_rel_diff(got[ok], ref[ok]).max()) if ok.any() else 0.0,
             "n_clause": n_clause, "max_abs": float(d.max()) if ok.any() else 0.0}
    if n_clause:
        assert scale is not None, f"{what}: {n_clause} outputs break the 1e-12/1e-15 rule, worst abs {d[~rule].max():.3e}"
        S = np.asarray(scale)[ok][~rule]
        worst = d[~rule] / S
        stats["max_d_over_S"] = float(worst.max())
        bad = worst > clause_rel
        assert not bad.any(), (f"{what}: {int(bad.sum())} outputs outside the conditioning clause, "
                               f"worst |d|/S = {worst.max():.3e}")
        assert n_clause <= max_clause_frac * max(1, ok.sum()), \
            f"{what}: {n_clause} of {int(ok.sum())} outputs needed the conditioning clause"
    return stats

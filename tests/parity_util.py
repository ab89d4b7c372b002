"""The parity criterion GPU-vs-oracle, written out once ("Tolerance").

north_star rule: |d| <= 1e-12 |ref|, or |d| <= 1e-15 where |ref| < 1e-3.
Conditioning clause: an output whose weighted stencil magnitude S dwarfs |ref| (a sign change
of xf inside the cell) carries rounding noise ~eps*S in ANY fp64 evaluation order, the oracle's
included; such an output passes if |d| <= 1e-12 * S, S from the oracle's scale helper.
The count of outputs that needed the clause is reported and bounded.

Every call appends one JSON line {test, n, max_eq1, n_rule_violations, n_clause, max_d_over_S} to
the parity log (PDFB_PARITY_LOG, default <repo>/gpurun_out/parity_log.jsonl), so that a run
leaves behind how many outputs needed the clause, test by test.
"""
import json
import os

import numpy as np

REL = 1e-12
ABS_SMALL = 1e-15
SMALL = 1e-3
EPS_EQ1 = 1e-16  # PAPER.md:87-91, eq. 1

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def parity_log_path():
    return os.environ.get("PDFB_PARITY_LOG", os.path.join(_ROOT, "gpurun_out", "parity_log.jsonl"))


def log_stats(what, stats):
    try:
        path = parity_log_path()
        os.makedirs(os.path.dirname(path), exist_ok=True)
        rec = {"test": os.environ.get("PYTEST_CURRENT_TEST", "").split(" ")[0], "what": what}
        rec.update(stats)
        with open(path, "a") as f:
            f.write(json.dumps(rec) + "\n")
    except OSError:
        pass  # a read-only tree must not fail a parity test


def eq1_rel_diff(got, ref):
    """r = |a - b| / (|b| + eps), eq. 1 of the paper."""
    return np.abs(got - ref) / (np.abs(ref) + EPS_EQ1)


def rule_violations(got, ref, slack=None):
    """Boolean mask of outputs that break the north_star rule (NaN patterns must agree).
    ``slack`` (same shape, >= 0) is added to the allowed |d| -- see check_parity."""
    d = np.abs(got - ref)
    r = np.abs(ref)
    sl = 0.0 if slack is None else np.asarray(slack)
    with np.errstate(invalid="ignore"):
        ok = np.where(r < SMALL, d <= ABS_SMALL + sl, d <= REL * r + sl)
    return ~ok & ~np.isnan(ref)


def check_parity(got, ref, scale=None, max_clause_frac=2e-3, what="", clause_rel=REL, log=True, slack=None):
    """Assert parity; returns a dict of statistics.

    ``slack`` (same shape as ``ref``, zero almost everywhere) is an extra |d| the CALLER derives for
    outputs where the result is a difference of nearly equal terms in the in-cell coordinate itself
    (xf -> 0 as t -> 1 on an x array of a handful of knots: DESIGN.md 5, "t -> 1"): such an output
    passes if |d| <= rule + slack.  How many outputs needed it is counted (``n_slack``) and logged.

    ``scale`` is the oracle's conditioning scale, same shape as ``ref`` -- or a callable
    ``scale(cols)`` that returns it for the listed point columns only (last axis of ``ref``), so
    that full-population checks pay for the scale helper on violators alone.
    ``clause_rel`` widens the conditioning clause only (never the north_star rule) for grids whose
    knots are much denser than the paper's: a last-bit difference in a coordinate logarithm moves
    t by ulp(u)/dU, so the clause scales with |u|/dU; the caller derives the factor."""
    got, ref = np.asarray(got), np.asarray(ref)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    nan_g, nan_r = np.isnan(got), np.isnan(ref)
    assert np.array_equal(nan_g, nan_r), f"{what}: NaN pattern differs"
    ok = ~nan_r
    n_ok = int(ok.sum())
    viol = rule_violations(got, ref, slack)
    n_clause = int(viol.sum())
    d = np.abs(got - ref)
    stats = {"n": n_ok, "max_eq1": float(eq1_rel_diff(got[ok], ref[ok]).max()) if n_ok else 0.0,
             "n_rule_violations": n_clause, "n_clause": n_clause, "max_abs": float(d[ok].max()) if n_ok else 0.0,
             "max_d_over_S": 0.0}
    if slack is not None:
        slack = np.broadcast_to(np.asarray(slack, dtype=np.float64), ref.shape)
        plain = rule_violations(got, ref)
        stats["n_slack"] = int((plain & ~viol).sum())          # outputs that pass only with the caller's slack
        used = plain & (slack > 0)
        stats["max_slack_used"] = float((d[used] / slack[used]).max()) if used.any() else 0.0
        d = np.maximum(d - slack, 0.0)                           # what the clause below still has to cover
    if n_clause:
        assert scale is not None, f"{what}: {n_clause} outputs break the 1e-12/1e-15 rule, worst abs {d[viol].max():.3e}"
        if callable(scale):
            cols = np.unique(np.nonzero(viol)[-1])
            sub = np.asarray(scale(cols))                  # [..., len(cols)]
            pos = np.searchsorted(cols, np.nonzero(viol)[-1])
            S = sub[np.nonzero(viol)[:-1] + (pos,)]
        else:
            S = np.asarray(scale)[viol]
        worst = d[viol] / S
        stats["max_d_over_S"] = float(worst.max())
        bad = worst > clause_rel
        if log:
            log_stats(what, stats)
        assert not bad.any(), (f"{what}: {int(bad.sum())} outputs outside the conditioning clause, "
                               f"worst |d|/S = {worst.max():.3e}")
        assert n_clause <= max_clause_frac * max(1, n_ok), \
            f"{what}: {n_clause} of {n_ok} outputs needed the conditioning clause"
    elif log:
        log_stats(what, stats)
    return stats


def merge_stats(parts):
    """Totals over chunks of one population."""
    tot = {"n": 0, "max_eq1": 0.0, "n_rule_violations": 0, "n_clause": 0, "max_abs": 0.0, "max_d_over_S": 0.0}
    for s in parts:
        for k in ("n", "n_rule_violations", "n_clause"):
            tot[k] += s[k]
        for k in ("max_eq1", "max_abs", "max_d_over_S"):
            tot[k] = max(tot[k], s[k])
    return tot


def check_parity_population(got_chunk, og, pids, x, q2, chunk=2_000_000, max_clause_frac=2e-3, what=""):
    """Parity on EVERY point of a batch ("parity is checked on all points"), in
    chunks: ``got_chunk(a, b)`` returns the library's [n_req, b-a] outputs for points a..b; the
    oracle runs on the same points, its scale helper only on the points that break the rule."""
    parts = []
    n = len(x)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        ref = og.xfxq2(pids, x[a:b], q2[a:b])
        xa, qa = x[a:b], q2[a:b]
        parts.append(check_parity(got_chunk(a, b), ref, lambda cols: og.xfxq2(pids, xa[cols], qa[cols], with_scale=True)[1],
                                  max_clause_frac=1.0, what=what, log=False))
    tot = merge_stats(parts)
    log_stats(what, tot)
    assert tot["n_clause"] <= max_clause_frac * max(1, tot["n"]), f"{what}: {tot}"
    return tot

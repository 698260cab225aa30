"""Pins of the PERM oracle. The supplement of the paper is not
available; the algorithm is Grassberger's (PRE 56, 3682 (1997)) with caller-given thresholds. What fixes it:
  * without population control a tour IS the pinned Rosenbluth chain of the same id (digest, weight, Ree2, Rg2);
  * forced enrichment / forced pruning at N = 3 have deterministic / two-valued outcomes computed by hand;
  * E[S] = c_n for ANY thresholds (unbiasedness) and the weighted <Ree2>, <Rg2> -> exact enumeration means
    (tests/golden/saw_cubic_exact.txt), 5 standard errors over tours;
  * tours are pure functions of (seed, tour id): sub-ranges reproduce, thresholds change the tour.
"""
import math

import numpy as np
import pytest

import oracle
from conftest import read_golden

INF = float("inf")


def exact(n):
    for row in read_golden("saw_cubic_exact.txt"):
        if int(row[0]) == n:
            return int(row[1]), int(row[2]), int(row[3])
    raise KeyError(n)


def thresholds(N, lo, hi):
    """ln_lo / ln_hi [N+1] around ln c_{n-1} (n = monomers): W in (lo c, hi c) is left alone."""
    counts = {int(r[0]): int(r[1]) for r in read_golden("saw_cubic_exact.txt")}
    ln_c = np.array([0.0, 0.0] + [math.log(counts[n - 1]) for n in range(2, N + 1)])
    return ln_c + math.log(lo), ln_c + math.log(hi), float(ln_c[N])


def test_no_population_control_is_the_rosenbluth_chain():
    for N, seed in ((8, 1), (16, 5), (40, 2)):
        lo, hi = np.full(N + 1, -INF), np.full(N + 1, INF)
        a = oracle.lattice_generate(N, 4000, seed)
        p = oracle.lattice_perm(N, 4000, seed, lo, hi, ln_ref=a.summary["ln_shift"])
        al = a.alive.astype(bool)
        assert np.array_equal(p.alive, a.alive)
        assert np.allclose(p.lnW[al], a.lnW[al], rtol=1e-13, atol=0) and np.all(np.isneginf(p.lnW[~al]))
        assert np.allclose(p.ree2[al], a.ree2[al], rtol=1e-13) and np.allclose(p.rg2[al], a.rg2[al], rtol=1e-13)
        assert p.summary["n_steps_attempted"] == a.summary["n_steps_attempted"]
        assert math.isclose(p.summary["mean_ree2"], a.summary["mean_ree2"], rel_tol=1e-12)
        assert math.isclose(p.summary["ln_mean_W"], a.summary["ln_mean_W"], rel_tol=1e-12)
        # same decisions: the tour's digest folds (m | event << 4, d) with event = 0, i.e. the chain's tokens
        assert np.array_equal(p.digest, a.digest)


def test_forced_enrichment_and_pruning_by_hand():
    N = 3
    lo, hi = np.full(N + 1, -INF), np.full(N + 1, INF)
    hi2 = hi.copy(); hi2[2] = math.log(5.9)                  # after step 1 W = 6 > 5.9: two copies of weight 3; each then has m = 5
    p = oracle.lattice_perm(N, 500, 3, lo, hi2, ln_ref=0.0)
    assert np.allclose(np.exp(p.lnW), 30.0, rtol=1e-13)      # 2 leaves x 15 = c_2, every tour
    assert p.summary["n_steps_attempted"] == 500 * 3 and math.isclose(p.summary["ln_mean_W"], math.log(30.0), rel_tol=1e-13)
    lo2 = lo.copy(); lo2[2] = math.log(6.1)                  # W = 6 < 6.1: killed with probability 1/2, else weight 12 -> leaf 60
    p = oracle.lattice_perm(N, 20000, 3, lo2, hi, ln_ref=0.0)
    W = np.where(p.alive == 1, np.exp(p.lnW), 0.0)
    assert set(np.round(W, 9)) == {0.0, 60.0}
    killed = int((W == 0).sum())
    assert abs(killed - 10000) < 5 * math.sqrt(20000 * 0.25)
    assert p.summary["n_dead"] == killed


@pytest.mark.parametrize("N,lo,hi", [(9, 0.5, 2.0), (13, 0.3, 3.0), (16, 0.9, 1.1), (16, 0.05, 1.5)])
def test_unbiased_for_any_thresholds(N, lo, hi):
    n = N - 1
    c, sr, sg = exact(n)
    ln_lo, ln_hi, ln_ref = thresholds(N, lo, hi)
    M = 60000
    p = oracle.lattice_perm(N, M, 11, ln_lo, ln_hi, ln_ref)
    assert (p.alive == 2).sum() == 0
    S = np.where(p.alive == 1, np.exp(p.lnW), 0.0)
    mean, se = S.mean(), S.std(ddof=1) / math.sqrt(M)
    assert abs(mean - c) < 5 * se, (mean, c, se)
    assert math.isclose(p.summary["ln_mean_W"], math.log(mean), rel_tol=1e-11)
    for arr, exact_mean, key in ((p.ree2, sr / c, "mean_ree2"), (p.rg2, sg / (N * N * c), "mean_rg2")):
        est = (S * arr).sum() / S.sum()
        se_r = math.sqrt(((S * (arr - est)) ** 2).sum()) / S.sum()
        assert abs(est - exact_mean) < 5 * se_r, (key, est, exact_mean, se_r)
        assert math.isclose(p.summary[key], est, rel_tol=1e-11)
    if hi / lo < 2.0:            # a narrow band must trigger enrichment and pruning
        assert p.summary["n_steps_attempted"] != M * n and p.summary["n_dead"] > 0


def test_variance_reduction_at_longer_chains():
    """Why PERM exists (the weight degeneracy of plain Rosenbluth sampling, SURVEY.md 8(d) config 4 note): at N = 100 the
    cost-normalised relative variance of the Z_N estimate must be clearly below the plain method's. Thresholds from the
    asymptotic form c_n ~ 1.21 mu^n n^(gamma - 1) (mu = 4.684, gamma = 1.157: control parameters only, any values are unbiased)."""
    N, M = 100, 4000
    n = np.arange(N + 1, dtype=np.float64) - 1.0
    ln_c = np.where(n >= 1, math.log(1.21) + n * math.log(4.684) + 0.157 * np.log(np.maximum(n, 1.0)), 0.0)
    p = oracle.lattice_perm(N, M, 4, ln_c + math.log(0.5), ln_c + math.log(2.0), float(ln_c[N]))
    a = oracle.lattice_generate(N, M, 4, outputs=("lnW", "alive"))
    assert (p.alive == 2).sum() == 0
    S = np.where(p.alive == 1, np.exp(p.lnW - ln_c[N]), 0.0)
    W = np.where(a.alive.astype(bool), np.exp(a.lnW - ln_c[N]), 0.0)
    eff_perm = S.var() / S.mean() ** 2 * p.summary["n_steps_attempted"]
    eff_ros = W.var() / W.mean() ** 2 * a.summary["n_steps_attempted"]
    assert eff_perm < 0.5 * eff_ros, (eff_perm, eff_ros)
    # and the two estimates of ln Z_N agree within their errors
    se_p = S.std(ddof=1) / math.sqrt(M) / S.mean(); se_r = W.std(ddof=1) / math.sqrt(M) / W.mean()
    assert abs(p.summary["ln_mean_W"] - a.summary["ln_mean_W"]) < 5 * math.hypot(se_p, se_r)


def test_tours_are_pure_functions_of_their_id():
    N = 14
    ln_lo, ln_hi, ln_ref = thresholds(N, 0.5, 2.0)
    p = oracle.lattice_perm(N, 3000, 9, ln_lo, ln_hi, ln_ref)
    q = oracle.lattice_perm(N, 1000, 9, ln_lo, ln_hi, ln_ref, tour_offset=1500)
    assert np.array_equal(p.digest[1500:2500], q.digest) and np.array_equal(p.lnW[1500:2500], q.lnW)
    r = oracle.lattice_perm(N, 3000, 9, ln_lo - 0.3, ln_hi, ln_ref)
    assert not np.array_equal(p.digest, r.digest)


def test_node_cap():
    N = 16
    _, _, ln_ref = thresholds(N, 0.5, 2.0)
    p = oracle.lattice_perm(N, 50, 2, np.full(N + 1, -INF), np.full(N + 1, -INF), ln_ref, max_nodes=2000)   # enrichment at every step
    assert (p.alive == 2).all() and p.summary["n_steps_attempted"] == 50 * 2000

"""Pins of the oracle's model path (other trial sets, Boltzmann-weighted trials).

What fixes it other than itself:
  * beta eps = 0, z = 6 must reproduce the pinned base oracle decision for decision (same digests);
  * SAW counts / Boltzmann sums of a pure-Python brute force written from the definitions (own direction lists);
  * the probabilities the step routine assigns to ALL enumerated walks sum to P_alive = 1 (non-statistical);
  * E[W] -> the enumerated (fixed-point) partition sum, W-weighted <Ree2> -> the exact Boltzmann mean (5 s.e.);
  * hand cases of the weights and of the fixed-point table.
"""
import itertools
import math

import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.filterwarnings("ignore")


def dirs(z):
    if z == 6:
        return [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    return [(dx, dy, dz) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1) if (dx, dy, dz) != (0, 0, 0)]


def adjacent(z, a, b):
    d = [abs(a[i] - b[i]) for i in range(3)]
    return sum(d) == 1 if z == 6 else (max(d) == 1)


def brute(n, z, q):
    """All n-step SAWs by plain product enumeration: count, sum q^contacts, sum q^contacts Ree2."""
    D = dirs(z)
    cnt, zsum, zr = 0, 0.0, 0.0
    for steps in itertools.product(range(z), repeat=n):
        r = [(0, 0, 0)]
        for d in steps:
            r.append(tuple(r[-1][i] + D[d][i] for i in range(3)))
        if len(set(r)) != n + 1:
            continue
        c = sum(1 for i in range(n + 1) for j in range(i + 2, n + 1) if adjacent(z, r[i], r[j]))
        cnt += 1; zsum += q ** c; zr += q ** c * sum(x * x for x in r[-1])
    return cnt, zsum, zr


def test_fixed_point_table():
    assert oracle.model_table(0.0) == [65536] * 32
    t = oracle.model_table(math.log(2.0))
    assert t[:8] == [65536 << c for c in range(8)]
    t = oracle.model_table(0.3)
    assert all(abs(t[c] / 65536.0 - math.exp(0.3 * c)) < 2.0 ** -17 * 1.0001 for c in range(32))


def test_beta0_z6_reproduces_base_oracle():
    for N, seed in ((16, 1), (40, 9)):
        a = oracle.lattice_generate(N, 3000, seed)
        b = oracle.lattice_model_generate(N, 3000, seed, z=6, beta_eps=0.0)
        assert np.array_equal(a.digest, b.digest) and np.array_equal(a.conf, b.conf) and np.array_equal(a.m_seq, b.m_seq)
        al = a.alive.astype(bool)
        assert np.allclose(a.lnW[al], b.lnW[al], rtol=1e-14, atol=0)
        assert math.isclose(a.summary["mean_ree2"], b.summary["mean_ree2"], rel_tol=1e-12)
        assert math.isclose(a.summary["ln_mean_W"], b.summary["ln_mean_W"], rel_tol=1e-12)


def test_hand_cases_weights():
    q = 0.5
    Q = oracle.model_table(q)
    # z = 6, U turn: r = (0,0,0),(1,0,0),(1,1,0): the trial -x from (1,1,0) lands on (0,1,0), neighbour of r_0 -> one contact
    w = oracle.lattice_model_step(np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0]]), 6, q)
    assert w == [Q[0], Q[1], Q[0], 0, Q[0], Q[0]]          # +x free, -x one contact, +y free, -y occupied (r_1), +z, -z
    # z = 26, second step from (1,0,0): the 26 sites around it; the origin is occupied; sites adjacent (Chebyshev 1) to the
    # origin, other than the head, make one contact
    w = oracle.lattice_model_step(np.array([[0, 0, 0], [1, 0, 0]]), 26, q)
    D = dirs(26)
    for d, e in enumerate(D):
        site = (1 + e[0], e[1], e[2])
        if site == (0, 0, 0):
            assert w[d] == 0
        else:
            assert w[d] == (Q[1] if max(abs(x) for x in site) == 1 else Q[0])


@pytest.mark.parametrize("z,n,beta", [(6, 4, 0.0), (6, 5, 0.4), (26, 2, 0.0), (26, 3, 0.3)])
def test_enumerator_against_brute_force(z, n, beta):
    q = math.exp(beta)
    cnt, zsum, zr = brute(n, z, q)
    e = oracle.saw_enumerate_model(n, z, beta)
    assert e["count"] == cnt
    assert math.isclose(e["sum_boltz"], zsum, rel_tol=1e-12) and math.isclose(e["sum_boltz_ree2"], zr, rel_tol=1e-12)
    assert math.isclose(e["sum_quant"], zsum, rel_tol=n * 2.0 ** -16)      # fixed-point factors: <= 2^-17 relative each


def test_counts_z26_and_z6():
    assert oracle.saw_enumerate_model(1, 26, 0.0)["count"] == 26
    assert oracle.saw_enumerate_model(2, 26, 0.0)["count"] == 26 * 25
    # z = 6 counts: the published series (tests/golden/saw_cubic_counts.txt is pinned elsewhere): c_5, c_6
    assert oracle.saw_enumerate_model(5, 6, 0.0)["count"] == 3534
    assert oracle.saw_enumerate_model(6, 6, 0.0)["count"] == 16926


@pytest.mark.parametrize("z,n,beta", [(6, 8, 0.5), (6, 7, 0.85), (26, 4, 0.0), (26, 4, 0.6)])
def test_step_probabilities_sum_to_one(z, n, beta):
    """sum over ALL n-step SAWs of prod_s w_s[d_s] / W_s = P_alive(n) = 1 (no trapped walk this short): a wrong contact
    count, a weight on an occupied site or a missing trial breaks the identity."""
    e = oracle.saw_enumerate_model(n, z, beta)
    assert math.isclose(e["sum_prob"], 1.0, rel_tol=1e-11)


@pytest.mark.parametrize("z,N,beta,seed", [(6, 8, 0.5, 3), (26, 5, 0.4, 4), (26, 4, 0.0, 5)])
def test_rosenbluth_estimates_converge(z, N, beta, seed):
    n = N - 1
    e = oracle.saw_enumerate_model(n, z, beta)
    M = 120000
    o = oracle.lattice_model_generate(N, M, seed, z=z, beta_eps=beta, outputs=("lnW", "ree2", "alive"))
    W = np.where(o.alive.astype(bool), np.exp(o.lnW), 0.0)
    mean, se = W.mean(), W.std(ddof=1) / math.sqrt(M)
    assert abs(mean - e["sum_quant"]) < 5 * se, (mean, e["sum_quant"], se)
    exact_ree2 = e["sum_boltz_ree2"] / e["sum_boltz"]
    est = (W * o.ree2).sum() / W.sum()
    # delta method s.e. of the ratio
    se_r = math.sqrt(((W * (o.ree2 - est)) ** 2).sum()) / W.sum()
    assert abs(est - exact_ree2) < 5 * se_r + 1e-4 * exact_ree2, (est, exact_ree2, se_r)
    assert math.isclose(o.summary["mean_ree2"], est, rel_tol=1e-10)
    assert math.isclose(o.summary["ln_mean_W"], math.log(mean), rel_tol=1e-10)


def test_invariants_z26():
    o = oracle.lattice_model_generate(24, 2000, 11, z=26, beta_eps=0.2)
    conf = o.conf.astype(np.int64)
    for i in range(0, 2000, 50):
        n_placed = 24 if o.alive[i] else int(np.count_nonzero(o.m_seq[i])) + 1
        r = conf[i, :n_placed]
        assert len({tuple(x) for x in r}) == n_placed                      # self-avoiding
        assert np.all(np.abs(np.diff(r, axis=0)).max(axis=1) == 1)        # every bond in the 26-neighbourhood
    assert o.m_seq[:, 0].min() == 26 and o.m_seq[:, 0].max() == 26 and o.m_seq[:, 1:].max() <= 25


def test_realspace_beta0_reproduces_base_and_well_counts():
    a = oracle.realspace_generate(20, 400, 16, 1.0, 1.0, 3)
    b = oracle.realspace_model_generate(20, 400, 16, 1.0, 1.0, 1.5, 0.0, 3)
    assert np.array_equal(a.digest, b.digest) and np.array_equal(a.conf, b.conf)
    # N = 3: the only earlier monomer a trial can see is r_0 at distance |r_1 + b u| with r_1 = b u_1: d2 = 2 b^2 (1 + cos);
    # inside the well (d < lambda sigma) and outside the core: weight q, else 1 -> E[W_2] / k = P(core free) + (q - 1) P(in well, free)
    k, lam, beta = 64, 1.5, 0.6
    o = oracle.realspace_model_generate(3, 40000, k, 1.0, 1.0, lam, beta, 5, outputs=("lnW", "alive"))
    W = np.where(o.alive.astype(bool), np.exp(o.lnW), 0.0) / k ** 2
    # P(d < x) for uniform direction: d^2 = 2(1 + c), c uniform on [-1,1] -> P(d^2 < x^2) = x^2 / 4
    p_core, p_well = 1.0 / 4, lam ** 2 / 4
    q = math.exp(beta)
    expect = (1 - p_well) + q * (p_well - p_core)
    se = W.std(ddof=1) / math.sqrt(len(W))
    assert abs(W.mean() - expect) < 5 * se + 1e-4, (W.mean(), expect, se)


def test_scaled_target_is_the_big_integer_quotient():
    """floor(u W / 2^32) (the selection threshold) against Python's exact integers, over both branches of
    the two-limb product: W < 2^32 (every z = 6 step) and W >= 2^32 (reached at z = 26, beta eps near 0.85), the carries
    at the limb boundary, and the extremes. A dropped high limb, a wrong shift or a missing carry fails here."""
    rng = np.random.default_rng(17)
    us = [0, 1, 2, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFE, 0xFFFFFFFF] + [int(v) for v in rng.integers(0, 1 << 32, 200)]
    Ws = [1, 2, 65536, 6 * 65536, (1 << 32) - 1, 1 << 32, (1 << 32) + 1, (1 << 33) - 1, 0x1_0000_FFFF, 0xFFFF_FFFF_FFFF,
          (1 << 62) + 12345, (1 << 63) - 1] + [int(v) for v in rng.integers(1, 1 << 62, 200)] \
         + [int(v) for v in rng.integers(1, 1 << 34, 200)]
    for u in us:
        for W in Ws:
            assert oracle.scaled_target(u, W) == (u * W) >> 32, (u, W)
    # the largest W a step can have: 26 free trials of 25 contacts each at beta eps = 0.85
    W = 26 * oracle.model_table(0.85)[25]
    assert W >= 1 << 32 and oracle.scaled_target(0xFFFFFFFF, W) == (0xFFFFFFFF * W) >> 32 < W


@pytest.mark.parametrize("k,seed", [(2, 41), (5, 42), (64, 43)])
def test_realspace_well_choice_is_boltzmann_proportional(k, seed):
    """Pins the CHOICE of oracle_realspace_model_generate (a trial is taken with probability Q[c_t] / W_s, Eq. 1-2
    PAPER.md:47-52), which the E[W] pin above cannot see. N = 3, b = 1: the bond-angle cosine c is uniform on [-1, 1] and
    Ree2 = 2 (1 + c); with t = 1 + c a trial overlaps for t < a = sigma^2 / 2 and sits in the well for t < w =
    (lambda sigma)^2 / 2, so the Boltzmann mean over the allowed directions is
        <Ree2> = [q (w^2 - a^2) + (4 - w^2)] / [q (w - a) + (2 - w)],  q = exp(beta eps),
    and the Rosenbluth estimator E[W Ree2] / E[W] equals it for ANY k when the choice is proportional to the weights.
    A uniform choice among the free trials gives something else (for large k: (4 - a^2) / (2 - a) = 2.5, the hard-sphere
    value), as does a choice by 1/weight or an off-by-one in the cumulative scan. The 2^-16 fixed point moves it by < 1e-5."""
    sigma, lam, beta = 1.0, 1.5, 0.6
    q = math.exp(beta)
    a, w = sigma ** 2 / 2, (lam * sigma) ** 2 / 2
    exact = (q * (w * w - a * a) + (4 - w * w)) / (q * (w - a) + (2 - w))
    assert math.isclose(exact, (1.015625 * q + 2.734375) / (0.625 * q + 0.875), rel_tol=1e-15) and abs(exact - 2.2767) < 1e-4
    M = 150000
    o = oracle.realspace_model_generate(3, M, k, 1.0, sigma, lam, beta, seed, outputs=("lnW", "ree2", "alive"))
    W = np.where(o.alive.astype(bool), np.exp(o.lnW), 0.0)
    est = (W * o.ree2).sum() / W.sum()
    se = math.sqrt(((W * (o.ree2 - est)) ** 2).sum()) / W.sum()          # delta method
    assert se < 0.01 and abs(est - exact) < 5 * se + 1e-4, (k, est, exact, se)
    assert abs(est - 2.5) > 10 * se                                       # the hard-sphere mean is resolved and excluded
    assert math.isclose(o.summary["mean_ree2"], est, rel_tol=1e-9)
    # q = 1 gives back the hard-sphere closed form 2.5 (survey pin P5) through the same code path
    o0 = oracle.realspace_model_generate(3, M, k, 1.0, sigma, lam, 0.0, seed, outputs=("lnW", "ree2", "alive"))
    W0 = np.where(o0.alive.astype(bool), np.exp(o0.lnW), 0.0)
    est0 = (W0 * o0.ree2).sum() / W0.sum()
    se0 = math.sqrt(((W0 * (o0.ree2 - est0)) ** 2).sum()) / W0.sum()
    assert abs(est0 - 2.5) < 5 * se0 + 1e-4, (est0, se0)

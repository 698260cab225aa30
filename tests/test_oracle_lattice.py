"""Pins for the lattice oracle (oracle/rosen_oracle.cpp) -- SURVEY.md 8(c) P1-P4.

Everything here checks the oracle against something other than itself: the published SAW
series, a brute-force enumeration with its own occupancy grid (C++, and a second tiny
pure-python one), exact rational identities, and invariants of the method.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle

E = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]])


def py_enumerate(n):
    """Independent pure-python DFS over n-step SAWs: count, sum Ree2, sum N^2 Rg2."""
    N = n + 1
    cnt = s_ree = s_rg = 0
    walk = [(0, 0, 0)]
    occ = {(0, 0, 0)}

    def rec():
        nonlocal cnt, s_ree, s_rg
        if len(walk) == N:
            cnt += 1
            x, y, z = walk[-1]
            s_ree += x * x + y * y + z * z
            sx = sum(p[0] for p in walk); sy = sum(p[1] for p in walk); sz = sum(p[2] for p in walk)
            s2 = sum(p[0] ** 2 + p[1] ** 2 + p[2] ** 2 for p in walk)
            s_rg += N * s2 - (sx * sx + sy * sy + sz * sz)
            return
        x, y, z = walk[-1]
        for dx, dy, dz in E:
            q = (x + dx, y + dy, z + dz)
            if q in occ:
                continue
            occ.add(q); walk.append(q)
            rec()
            walk.pop(); occ.remove(q)

    rec()
    return cnt, s_ree, s_rg


def test_enumerator_matches_published_counts(golden):
    counts = {int(n): int(c) for n, c in golden("saw_cubic_counts.txt")}
    for n in range(1, 10):
        assert oracle.saw_enumerate(n)["count"] == counts[n]
    assert oracle.saw_enumerate(10, fix_first=True)["count"] == counts[10]
    assert counts[3] == 6 * 5 * 5 and counts[4] == 6 * 5 ** 3 - 24


def test_enumerator_matches_python_bruteforce():
    for n in range(1, 7):
        e = oracle.saw_enumerate(n)
        assert (e["count"], e["sum_ree2"], e["sum_n2rg2"]) == py_enumerate(n)
    # hand values: n=1 Ree2=1; n=2: 6 straight (4) + 24 bent (2)
    assert oracle.saw_enumerate(2)["sum_ree2"] == 6 * 4 + 24 * 2


def test_exact_golden_file_consistent(golden):
    counts = {int(n): int(c) for n, c in golden("saw_cubic_counts.txt")}
    rows = golden("saw_cubic_exact.txt")
    assert len(rows) >= 12
    for n, c, _, _, pa in rows:
        assert int(c) == counts[int(n)]
        num, den = (int(x) for x in pa.split("/"))
        if int(n) <= 11:
            assert num == den == 1
    row12 = [r for r in rows if r[0] == "12"][0]
    # first trapped walks: 240 walks of 11 steps, each generated with probability 1/(6*5^10)
    assert 1 - Fraction(*[int(x) for x in row12[4].split("/")]) == Fraction(240, 6 * 5 ** 10)


@pytest.mark.parametrize("n", [4, 7, 10])
def test_free_site_routine_exact_survival_identity(n):
    """P3: sum over ALL n-step SAWs of 1/W(w), W from the oracle's free-site routine, is exactly 1
    (no walk of <= 11 steps can be trapped). A wrong count anywhere changes the rational sum."""
    e = oracle.saw_enumerate(n, fix_first=(n >= 9))
    total = sum(Fraction(c, 2 ** a * 3 ** b * 5 ** cc) for (a, b, cc), c in e["hist"].items())
    assert total == 1
    assert sum(e["hist"].values()) == e["count"]


def test_free_dirs_hand_cases():
    assert oracle.lattice_free_dirs(np.array([[0, 0, 0]])) == [0, 1, 2, 3, 4, 5]          # m_1 = 6
    assert oracle.lattice_free_dirs(np.array([[0, 0, 0], [1, 0, 0]])) == [0, 2, 3, 4, 5]  # back site -x
    # U-turn: (0,0,0),(1,0,0),(1,1,0),(0,1,0): head (0,1,0); -x free, +x = predecessor, -y = origin
    assert oracle.lattice_free_dirs(np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0], [0, 1, 0]])) == [1, 2, 4, 5]
    # planar loop around the origin: head (-1,0,0) has +x = origin (occupied, j=0) and -z = its predecessor
    loop = np.array([[0, 0, 0], [0, 0, 1], [1, 0, 1], [1, 0, 0], [1, 0, -1], [0, 0, -1], [-1, 0, -1], [-1, 0, 0]])
    assert oracle.lattice_free_dirs(loop) == [1, 2, 3, 4]
    # shortest trap (11 steps): visit the five other neighbours of T = (0,0,0), then step into T
    trap = np.array([[1, 0, 0], [1, 1, 0], [0, 1, 0], [-1, 1, 0], [-1, 0, 0], [-1, 0, 1], [0, 0, 1], [0, -1, 1],
                     [0, -1, 0], [0, -1, -1], [0, 0, -1], [0, 0, 0]])
    assert oracle.lattice_free_dirs(trap) == []          # m = 0: dead end
    assert oracle.lattice_free_dirs(trap[:-1]) == [0, 1, 2, 4, 5]   # one step earlier only -y (predecessor) is taken


def _weighted_stats(r):
    """Weighted means and their standard errors from per-chain arrays (dead chains: w = 0)."""
    lnw = np.where(r.alive == 1, r.lnW, -np.inf)
    L = r.summary["ln_shift"]
    w = np.exp(lnw - L)
    n = w.size
    mean_w = w.mean()
    se_w = w.std(ddof=1) / math.sqrt(n)
    out = {"lnmeanW": L + math.log(mean_w), "rel_se_W": se_w / mean_w}
    for name, a in (("ree2", r.ree2), ("rg2", r.rg2)):
        ratio = (w * a).sum() / w.sum()
        # delta-method s.e. of a ratio estimator
        resid = w * (a - ratio)
        out[name] = ratio
        out[name + "_se"] = resid.std(ddof=1) / math.sqrt(n) / mean_w
    return out


@pytest.mark.parametrize("N,n_chains,seed", [(4, 1 << 15, 5), (8, 1 << 16, 2), (11, 1 << 17, 3), (16, 1 << 17, 1)])
def test_rosenbluth_estimates_converge_to_enumeration(golden, N, n_chains, seed):
    """P1 + P2: E[W_N] = c_n (Eq. 3/6) and the W-weighted averages (Eq. 2) equal the uniform-SAW
    means from exact enumeration, within 5 standard errors."""
    n = N - 1
    row = [r for r in golden("saw_cubic_exact.txt") if int(r[0]) == n][0]
    c_n, s_ree, s_rg = int(row[1]), int(row[2]), int(row[3])
    r = oracle.lattice_generate(N, n_chains, seed)
    st = _weighted_stats(r)
    assert abs(math.exp(st["lnmeanW"] - math.log(c_n)) - 1) <= 5 * st["rel_se_W"] + 1e-12   # N=4: W = 150 always
    assert abs(st["ree2"] - s_ree / c_n) < 5 * st["ree2_se"]
    assert abs(st["rg2"] - s_rg / (N * N * c_n)) < 5 * st["rg2_se"]
    # the summary is the same estimator
    assert math.isclose(r.summary["mean_ree2"], st["ree2"], rel_tol=1e-12)
    assert math.isclose(r.summary["mean_rg2"], st["rg2"], rel_tol=1e-12)
    assert math.isclose(r.summary["ln_mean_W"], st["lnmeanW"], rel_tol=1e-12)


def test_invariants_P4():
    N, n_chains = 48, 4096
    r = oracle.lattice_generate(N, n_chains, 11)
    m = r.m_seq.astype(int)
    assert np.all(m[:, 0] == 6)                                   # m_1 = 6 (Alg. 1 line 7, p <- 1/6)
    assert m[:, 1:].max() <= 5 and m.min() >= 0
    dead = r.alive == 0
    assert dead.sum() == r.summary["n_dead"] and dead.sum() > 0    # attrition ~1e-3 at N=48
    assert np.all(np.isneginf(r.lnW[dead])) and np.all(np.isfinite(r.lnW[~dead]))
    assert np.all((m == 0).any(axis=1) == dead)                   # dead <=> some m_s = 0
    steps = np.where(dead, (m == 0).argmax(axis=1) + 1, N - 1)
    assert steps.sum() == r.summary["n_steps_attempted"]
    for i in range(n_chains):
        conf = r.conf[i]
        L = steps[i] if not dead[i] else steps[i] - 1             # bonds actually placed
        bonds = np.abs(np.diff(conf[: L + 1], axis=0)).sum(axis=1)
        assert np.all(bonds == 1)                                  # unit steps
        assert len({tuple(p) for p in conf[: L + 1]}) == L + 1     # self-avoiding
        assert np.all(conf[L + 1:] == 0)                           # zero-filled after death
        assert np.all(m[i, steps[i]:] == 0)
    alive = ~dead
    lnw = np.log(np.where(m[alive] > 0, m[alive], 1)).sum(axis=1)
    assert np.allclose(r.lnW[alive], lnw, rtol=1e-13)              # W = prod m_s (Eq. 3)
    ree2 = (r.conf[:, -1, :].astype(np.int64) ** 2).sum(axis=1)
    assert np.all(r.ree2[alive] == ree2[alive]) and np.all(r.ree2[dead] == 0)
    c = r.conf.astype(np.float64)
    rg2 = ((c - c.mean(axis=1, keepdims=True)) ** 2).sum(axis=2).mean(axis=1)
    assert np.allclose(r.rg2[alive], rg2[alive], rtol=1e-12)
    # dead chains are kept in the denominators
    assert r.summary["n_chains"] == n_chains
    assert math.isclose(r.summary["attrition"], dead.mean())


def test_chain_offset_and_seed_reproducibility():
    a = oracle.lattice_generate(20, 512, 9, chain_offset=0)
    b = oracle.lattice_generate(20, 256, 9, chain_offset=256)
    assert np.array_equal(a.conf[256:], b.conf) and np.array_equal(a.digest[256:], b.digest)
    c = oracle.lattice_generate(20, 512, 10)
    assert not np.array_equal(a.conf, c.conf)
    big = oracle.lattice_generate(20, 4, 9, chain_offset=(1 << 32) - 2)   # chain id crosses 2^32
    lo = oracle.lattice_generate(20, 4, 9, chain_offset=0)
    assert not np.array_equal(big.conf[2:], lo.conf[:2])


def test_selection_rule_and_direction_order():
    """The chosen site is the sel-th free direction in the order +x,-x,+y,-y,+z,-z with
    sel = (u*m)>>32, u = Philox word (chain, s): recomputed here from the documented keying."""
    N, seed = 12, 77
    r = oracle.lattice_generate(N, 64, seed, chain_offset=5)
    for i in range(64):
        chain = 5 + i
        for s in range(1, N):
            if r.m_seq[i, s - 1] == 0:
                break
            free = oracle.lattice_free_dirs(r.conf[i, :s])
            assert len(free) == r.m_seq[i, s - 1]
            u = oracle.philox4x32_10((chain & 0xFFFFFFFF, chain >> 32, s >> 2, 0), (seed, 0))[s & 3]
            d = free[(u * len(free)) >> 32]
            assert np.array_equal(r.conf[i, s] - r.conf[i, s - 1], E[d])


def test_digest_definition():
    N = 10
    r = oracle.lattice_generate(N, 32, 3)
    for i in range(32):
        h = 0xCBF29CE484222325
        for s in range(1, N):
            m = int(r.m_seq[i, s - 1])
            if m == 0:
                h = ((h ^ (0 | 0xFF << 8)) * 0x100000001B3) & (2 ** 64 - 1)
                break
            d = int(np.flatnonzero((E == (r.conf[i, s] - r.conf[i, s - 1])).all(axis=1))[0])
            h = ((h ^ (m | d << 8)) * 0x100000001B3) & (2 ** 64 - 1)
        assert h == int(r.digest[i])
    assert int(np.bitwise_xor.reduce(r.digest)) == r.summary["digest_xor"]
    assert int(r.digest.sum(dtype=np.uint64)) == r.summary["digest_sum"]


def test_invalid_arguments():
    with pytest.raises(ValueError):
        oracle.lattice_generate(1, 4, 0)
    with pytest.raises(ValueError):
        oracle.lattice_generate(8, 0, 0)


def test_long_chain_shift_cancels_and_is_added_back():
    """Reading A18: for N > 512 the oracle normalises with L = the largest lnW of the run (the fixed
    bound ln6 + (N-2) ln5 underflows fp64 at N ~ 10^4). L must cancel in Eq. 2 and be added back in Eq. 6: the summary
    equals a log-sum-exp computed here from the per-chain lnW, and the N = 512 / 513 pair brackets the switch."""
    for N in (512, 513, 1500, 6000):
        r = oracle.lattice_generate(N, 300 if N < 6000 else 60, 31)
        S = r.summary
        a = r.alive == 1
        lnw = r.lnW[a]
        top = lnw.max()
        if N <= 512:
            assert math.isclose(S["ln_shift"], math.log(6.0) + (N - 2) * math.log(5.0), rel_tol=1e-15)
        else:
            assert S["ln_shift"] == top
            assert S["sum_w"] >= 1.0 and S["sum_w2"] >= 1.0            # the heaviest chain has w = 1 exactly
        rel = np.exp(lnw - top)
        assert math.isclose(S["ln_mean_W"], top + math.log(rel.sum() / r.alive.size), rel_tol=1e-12)
        assert math.isclose(S["mean_ree2"], float((rel * r.ree2[a]).sum() / rel.sum()), rel_tol=1e-12)
        assert math.isclose(S["mean_rg2"], float((rel * r.rg2[a]).sum() / rel.sum()), rel_tol=1e-12)
        assert S["n_dead"] == int((~a).sum()) and 0 < S["sum_w"] < float("inf") and S["sum_w2"] > 0
    # no chain alive: L = 0, sums 0, means 0/0
    r = oracle.lattice_generate(16383, 3, 20)
    assert r.summary["n_dead"] == 3 and r.summary["ln_shift"] == 0.0 and r.summary["sum_w"] == 0.0
    assert math.isnan(r.summary["mean_ree2"])

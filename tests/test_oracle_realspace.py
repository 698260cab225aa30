"""Pins for the real-space oracle (oracle/rosen_oracle.cpp) -- SURVEY.md 8(c) P4-P6 and the
unit-sphere direction map."""
import math

import numpy as np
import pytest

import oracle


# ------------------------------------------------------------------ direction map ("rngonsphere")
def exact_direction(wz, wphi):
    """The map DESIGN.md 3.3 defines, evaluated in fp64 with libm (independent of the polynomials)."""
    z = ((2 * (wz >> 9) + 1) - 2 ** 23) / 2.0 ** 23
    a = wphi >> 8
    phi = (2 * a + 1) / 2.0 ** 25 * 2.0 * math.pi          # midpoint of cell a of 2^24 on [0, 2pi)
    rho = math.sqrt(1.0 - z * z)
    return np.array([rho * math.cos(phi), rho * math.sin(phi), z])


def test_direction_against_libm():
    rng = np.random.default_rng(12345)
    words = rng.integers(0, 2 ** 32, size=(20000, 2), dtype=np.uint64)
    worst = 0.0
    for wz, wphi in words:
        u = oracle.direction(int(wz), int(wphi)).astype(np.float64)
        worst = max(worst, np.abs(u - exact_direction(int(wz), int(wphi))).max())
        assert abs(np.dot(u, u) - 1.0) < 4e-7
    assert worst < 2.5e-7          # ~2 ulp of fp32 at 1.0


def test_direction_octants_and_edges():
    # every octant, first / last / middle cell: quadrant signs, mirroring and swap are all visible here
    for oct_ in range(8):
        for f in (0, 1, 0x0FFFFF, 0x100000, 0x1FFFFE, 0x1FFFFF):
            a = (oct_ << 21) | f
            for low in (0, 0xFF):
                wphi = (a << 8) | low                      # low 8 bits are ignored
                for wz in (0, 0x1FF, 0x80000000, 0xFFFFFFFF, 0x7FFFFFFF):
                    u = oracle.direction(wz, wphi).astype(np.float64)
                    assert np.abs(u - exact_direction(wz, wphi)).max() < 2.5e-7
    # z is exact: symmetric midpoints, never +-1
    assert oracle.direction(0, 0)[2] == np.float32(-1 + 2.0 ** -23)
    assert oracle.direction(0xFFFFFFFF, 0)[2] == np.float32(1 - 2.0 ** -23)
    assert oracle.direction(0x80000000, 0)[2] == np.float32(2.0 ** -23)


def test_direction_azimuth_monotone():
    a = np.arange(0, 2 ** 24, 4099, dtype=np.int64)
    phi = np.array([math.atan2(*oracle.direction(0x80000000, int(x) << 8)[[1, 0]].astype(float)) for x in a])
    phi = np.mod(phi, 2 * math.pi)
    assert np.all(np.diff(phi) > 0)


def test_direction_moments():
    rng = np.random.default_rng(7)
    n = 40000
    words = rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64)
    U = np.array([oracle.direction(int(a), int(b)) for a, b in words], dtype=np.float64)
    assert np.all(np.abs(U.mean(axis=0)) < 5 * math.sqrt(1 / 3 / n))
    C = U.T @ U / n
    assert np.all(np.abs(C - np.eye(3) / 3) < 5 * math.sqrt(0.1 / n))


# ------------------------------------------------------------------ grower
def _weighted(r):
    w = np.where(r.alive == 1, np.exp(r.lnW - r.summary["ln_shift"]), 0.0)
    out = {}
    for name, a in (("ree2", r.ree2), ("rg2", r.rg2)):
        ratio = (w * a).sum() / w.sum()
        resid = w * (a - ratio)
        out[name] = ratio
        out[name + "_se"] = resid.std(ddof=1) / math.sqrt(w.size) / w.mean()
    return out


@pytest.mark.parametrize("sigma,frac,ree2,rg2", [(1.0, 0.75, 2.5, 0.5), (0.8, 0.84, 2.32, 0.48)])
def test_closed_forms_three_monomers_P5(sigma, frac, ree2, rg2):
    """N = 3, b = 1: monomer 2 must stay outside the sphere of monomer 0, i.e.
    cos(gamma) >= sigma^2/(2 b^2) - 1 =: c0 for the bond angle; with a uniform direction the free
    fraction is (1-c0)/2, <Ree2> = 2 b^2 (1 + (1+c0)/2), <Rg2> = (2 b^2 + <Ree2>) / 9 ... all exact."""
    k, n_chains = 16, 1 << 16
    c0 = sigma * sigma / 2.0 - 1.0
    assert math.isclose(frac, (1 - c0) / 2) and math.isclose(ree2, 2 * (1 + (1 + c0) / 2))
    assert math.isclose(rg2, (1 + 1 + ree2) / 9)          # Rg2 = sum_{i<j} r_ij^2 / N^2
    r = oracle.realspace_generate(3, n_chains, k, 1.0, sigma, 3)
    m2 = r.m_seq[:, 1].astype(float)
    assert np.all(r.m_seq[:, 0] == k)                      # nothing to test at step 1
    assert abs(m2.mean() / k - frac) < 5 * math.sqrt(frac * (1 - frac) / (k * n_chains))
    # m_2 ~ Binomial(k, frac): variance check
    assert abs(m2.var() - k * frac * (1 - frac)) < 0.05 * k * frac * (1 - frac)
    st = _weighted(r)
    assert abs(st["ree2"] - ree2) < 5 * st["ree2_se"]
    assert abs(st["rg2"] - rg2) < 5 * st["rg2_se"]


def test_freely_jointed_chain_P6():
    N, k, b, n_chains = 64, 16, 1.5, 4096
    r = oracle.realspace_generate(N, n_chains, k, b, 0.0, 21)
    assert np.all(r.m_seq == k) and np.all(r.alive == 1)
    assert np.allclose(r.lnW, (N - 1) * math.log(k), rtol=1e-14)
    assert math.isclose(r.summary["ln_mean_W"], (N - 1) * math.log(k), rel_tol=1e-13)
    se = r.ree2.std(ddof=1) / math.sqrt(n_chains)
    assert abs(r.ree2.mean() - (N - 1) * b * b) < 5 * se
    seg = r.rg2.std(ddof=1) / math.sqrt(n_chains)
    assert abs(r.rg2.mean() - b * b * (N * N - 1) / (6 * N)) < 5 * seg
    assert math.isclose(r.summary["mean_ree2"], r.ree2.mean(), rel_tol=1e-12)


def test_invariants_P4():
    N, k, b, sigma, n_chains = 32, 8, 1.0, 1.0, 1024
    r = oracle.realspace_generate(N, n_chains, k, b, sigma, 5)
    dead = r.alive == 0
    assert dead.sum() == r.summary["n_dead"] and dead.sum() > 0
    m = r.m_seq.astype(int)
    assert np.all(m[:, 0] == k) and m.max() <= k
    assert np.all((m == 0).any(axis=1) == dead)
    steps = np.where(dead, (m == 0).argmax(axis=1) + 1, N - 1)
    assert steps.sum() == r.summary["n_steps_attempted"]
    for i in range(n_chains):
        L = steps[i] - 1 if dead[i] else steps[i]
        c = r.conf[i, : L + 1].astype(np.float64)
        assert np.allclose(np.linalg.norm(np.diff(c, axis=0), axis=1), b, atol=2e-5)
        d = np.linalg.norm(c[:, None, :] - c[None, :, :], axis=2)
        iu = np.triu_indices(L + 1, 2)                     # non-bonded pairs j < i-1
        assert np.all(d[iu] >= sigma * (1 - 1e-5))
        assert np.all(r.conf[i, L + 1:] == 0) and np.all(m[i, steps[i]:] == 0)
    alive = ~dead
    assert np.allclose(r.lnW[alive], np.log(m[alive]).sum(axis=1), rtol=1e-13)
    assert np.all(np.isneginf(r.lnW[dead]))
    c = r.conf.astype(np.float64)
    assert np.allclose(r.ree2[alive], (c[alive, -1] ** 2).sum(axis=1), rtol=1e-14)
    rg2 = ((c - c.mean(axis=1, keepdims=True)) ** 2).sum(axis=2).mean(axis=1)
    assert np.allclose(r.rg2[alive], rg2[alive], rtol=1e-12)


def _fmaf(a, b, c):
    return np.float32(np.float64(a) * np.float64(b) + np.float64(c))


def test_keying_selection_and_overlap_rule():
    """Re-derive every step of a few chains from the documented keying (DESIGN.md 3.1/3.3):
    trial t of step s uses block (chain, s, 1+(t>>1)), words (0,1) / (2,3); the selection word is
    word s&3 of block (chain, s>>2, 0); overlap is d2 < sigma^2 against j <= s-2 (strict, A11)."""
    N, k, b, sigma, seed, off = 10, 6, np.float32(1.0), np.float32(0.9), 42, 3
    r = oracle.realspace_generate(N, 16, k, float(b), float(sigma), seed, chain_offset=off)
    s2 = np.float32(sigma * sigma)
    for i in range(16):
        chain = off + i
        for s in range(1, N):
            if r.m_seq[i, s - 1] == 0:
                break
            head = r.conf[i, s - 1]
            free = []
            for t in range(k):
                blk = oracle.philox4x32_10((chain, 0, s, 1 + (t >> 1)), (seed, 0))
                u = oracle.direction(blk[2 * (t & 1)], blk[2 * (t & 1) + 1])
                trial = np.array([_fmaf(b, u[a], head[a]) for a in range(3)], dtype=np.float32)
                ok = True
                for j in range(s - 1):
                    d = r.conf[i, j] - trial
                    d2 = _fmaf(d[2], d[2], _fmaf(d[1], d[1], np.float32(d[0] * d[0])))
                    if d2 < s2:
                        ok = False
                if ok:
                    free.append(trial)
            assert len(free) == r.m_seq[i, s - 1]
            u32 = oracle.philox4x32_10((chain, 0, s >> 2, 0), (seed, 0))[s & 3]
            assert np.array_equal(free[(u32 * len(free)) >> 32], r.conf[i, s])


def test_offset_reproducibility_and_arguments():
    a = oracle.realspace_generate(12, 64, 8, 1.0, 1.0, 9)
    b = oracle.realspace_generate(12, 32, 8, 1.0, 1.0, 9, chain_offset=32)
    assert np.array_equal(a.conf[32:], b.conf) and np.array_equal(a.digest[32:], b.digest)
    for bad in [dict(N=1), dict(k=0), dict(k=256), dict(b=0.0), dict(sigma=-1.0), dict(b=float("nan"))]:
        args = dict(N=8, n=4, k=4, b=1.0, sigma=1.0)
        args.update(bad)
        with pytest.raises(ValueError):
            oracle.realspace_generate(args["N"], args["n"], args["k"], args["b"], args["sigma"], 0)


def test_scaling_exponent_consistency_P10():
    """nu from <Ree2> ~ (N-1)^(2 nu): lattice and real space agree (north_star)."""
    Ns = (8, 16, 32)
    lat = [oracle.lattice_generate(N, 1 << 14, 11, outputs=()).summary["mean_ree2"] for N in Ns]
    rs = [oracle.realspace_generate(N, 1 << 11, 8, 1.0, 1.0, 11, outputs=()).summary["mean_ree2"] for N in Ns]
    x = np.log(np.array(Ns) - 1.0)
    nu_lat = np.polyfit(x, np.log(lat), 1)[0] / 2
    nu_rs = np.polyfit(x, np.log(rs), 1)[0] / 2
    assert 0.56 < nu_lat < 0.64 and 0.56 < nu_rs < 0.66
    assert abs(nu_lat - nu_rs) < 0.05


def test_long_chain_shift_is_the_largest_lnW():
    """Reading A18 for real space (N > 2048): L = max lnW instead of (N-1) ln k, which underflows exp(lnW - L) for
    chains of 10^4 monomers (lnW - (N-1) ln k ~ N ln(free fraction)). Checked against a shift-free log-sum-exp."""
    for N, k, sigma in ((2048, 4, 0.3), (2049, 4, 0.3)):
        r = oracle.realspace_generate(N, 6, k, 1.0, sigma, 5)
        S = r.summary
        a = r.alive == 1
        assert a.any()
        top = r.lnW[a].max()
        if N <= 2048:
            assert math.isclose(S["ln_shift"], (N - 1) * math.log(k), rel_tol=1e-15)
        else:
            assert S["ln_shift"] == top and S["sum_w"] >= 1.0
        rel = np.exp(r.lnW[a] - top)
        assert math.isclose(S["ln_mean_W"], top + math.log(rel.sum() / a.size), rel_tol=1e-12)
        assert math.isclose(S["mean_ree2"], float((rel * r.ree2[a]).sum() / rel.sum()), rel_tol=1e-12)

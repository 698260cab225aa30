"""Scaling analysis (Eq. 4-7): oracle pins and C-ABI parity (host function)."""
import math

import numpy as np
import pytest

import oracle


def synthetic(Ns, a, nu, mu, gamma, c, steps=True):
    x = np.asarray(Ns, dtype=np.float64) - (1.0 if steps else 0.0)
    return a * x ** (2 * nu), c + x * math.log(mu) + (gamma - 1.0) * np.log(x)


def test_oracle_recovers_exact_power_laws():
    Ns = [8, 16, 32, 64, 128, 256]
    for steps in (True, False):
        r2, lz = synthetic(Ns, 1.23, 0.5876, 4.684, 1.1568, 0.3, steps)
        f = oracle.fit_exponents(Ns, r2, lz, use_steps=steps)
        assert abs(f["nu"] - 0.5876) < 1e-12 and abs(f["mu"] - 4.684) < 1e-10 and abs(f["gamma"] - 1.1568) < 1e-9
        assert abs(f["ln_a"] - math.log(1.23)) < 1e-11 and abs(f["c"] - 0.3) < 1e-9


def test_oracle_on_exact_enumeration_counts(golden):
    """Z_n = c_n exactly (tests/golden/saw_cubic_counts.txt, n = 1..12 steps): the three-parameter fit of Eq. 7 on these
    short walks lands near the literature values quoted in the paper's Table 4 (mu 4.684, gamma 1.1608)
    within the known finite-size drift, and the random walk c_n = 6^n gives mu = 6, gamma = 1 exactly."""
    rows = [(int(r[0]), int(r[1])) for r in golden("saw_cubic_counts.txt")]
    rows = [r for r in rows if 4 <= r[0] <= 12]
    n = [r[0] for r in rows]
    f = oracle.fit_exponents([k + 1 for k in n], [1.0 + k for k in n], [math.log(c) for _, c in rows], use_steps=True)
    assert 4.60 < f["mu"] < 4.75 and 1.10 < f["gamma"] < 1.30
    g = oracle.fit_exponents([k + 1 for k in n], [float(k) for k in n], [k * math.log(6.0) for k in n])
    assert abs(g["mu"] - 6.0) < 1e-9 and abs(g["gamma"] - 1.0) < 1e-9 and abs(g["nu"] - 0.5) < 1e-12


def test_cabi_fit_matches_oracle():
    import paper_1704_04381_b200 as R
    from paper_1704_04381_b200 import build
    build.build()
    rng = np.random.default_rng(5)
    Ns = [8, 16, 32, 64, 128, 256]
    r2, lz = synthetic(Ns, 0.9, 0.6, 4.69, 1.16, -0.2)
    r2 = r2 * np.exp(rng.normal(0, 0.01, len(Ns))); lz = lz + rng.normal(0, 0.02, len(Ns))
    for steps in (True, False):
        a = R.rosen_fit_exponents(Ns, r2, lz, use_steps=steps)
        b = oracle.fit_exponents(Ns, r2, lz, use_steps=steps)
        for k in ("nu", "ln_a", "mu", "gamma", "c"):
            assert math.isclose(a[k], b[k], rel_tol=1e-9, abs_tol=1e-9), (k, a[k], b[k])
        assert a["rms_ree2"] > 0 and a["rms_lnZ"] > 0
    two = R.rosen_fit_exponents([8, 64], [10.9, 152.9], [1.0, 2.0])
    assert math.isnan(two["mu"]) and math.isclose(two["nu"], 0.5 * math.log(152.9 / 10.9) / math.log(63 / 7), rel_tol=1e-12)
    for bad in (([8], [1.0], [1.0]), ([8, 1], [1.0, 2.0], [1.0, 2.0]), ([8, 16], [1.0, -2.0], [1.0, 2.0]), ([8, 8, 8], [1.0] * 3, [1.0] * 3)):
        with pytest.raises(R.RosenError):
            R.rosen_fit_exponents(*bad)

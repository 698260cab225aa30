"""GPU parity on WHOLE populations at the sizes BASELINE.json quotes.

One GPU call in the launch configuration bench.py times is compared with the unchanged single-thread oracle run
over the same chain ids on all host cores (tests/oracle_pool.py):
  lattice     digest_xor, digest_sum, n_dead, n_steps_attempted exact; ensemble sums within 1e-12 relative
  real space  per-chain digests compared one by one -> flip fraction (bar 1e-4, expected 0); sums within 1e-6
The oracle does ~9e5 lattice chains/s (N = 64) on 16 cores: config 2 costs ~20 s, config 3 ~50 s, config 4's N = 128 point ~70 s.
Every test compares the population its name states, however long the host takes, and asserts the count it compared. Only
with FULLPOP_ALLOW_CUT=1 in the environment (a slow development box) may a population be cut to the largest power-of-two
prefix that fits FULLPOP_BUDGET_S; the test then warns, and still covers the prefix through the same launch geometry.
"""
import math
import os
import time
import warnings

import numpy as np
import pytest

from oracle_pool import SUM_KEYS, host_threads, oracle_population, oracle_workload_arrays
from paper_1704_04381_b200 import workloads

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

BUDGET_S = float(os.environ.get("FULLPOP_BUDGET_S", "150"))


@pytest.fixture(scope="module")
def R():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1704_04381_b200 as R
    R.load_library()
    return R


ALLOW_CUT = os.environ.get("FULLPOP_ALLOW_CUT", "") == "1"


def affordable(kind, N, n_chains, seed, **kw):
    """n_chains -- the whole population -- unless FULLPOP_ALLOW_CUT=1, in which case the largest power-of-two population
    <= n_chains whose oracle run fits the budget on this host."""
    if not ALLOW_CUT:
        return n_chains
    probe = 256 if (kind == "lattice" and N <= 64) else 32
    t0 = time.perf_counter()
    oracle_population(kind, N, probe * host_threads(), seed, ranges_per_thread=1, **kw)
    rate = probe * host_threads() / max(time.perf_counter() - t0, 1e-6)
    n = n_chains
    while n > 4096 and n / rate > BUDGET_S:
        n //= 2
    if n != n_chains:
        warnings.warn(f"[fullpop] {kind} N={N}: FULLPOP_ALLOW_CUT=1 and the host does {rate:.3g} chains/s on {host_threads()} "
                      f"threads: population cut {n_chains} -> {n}")
    return n


def compared(n, n_chains):
    """Every test ends here: the count that was compared is the count the test names (or a cut was explicitly allowed)."""
    assert n == n_chains or ALLOW_CUT, f"compared {n} of {n_chains} chains"
    assert n >= min(n_chains, 4096)


def check_lattice(R, N, n_chains, seed, rel=1e-12):
    n = affordable("lattice", N, n_chains, seed)
    s, _ = R.rosen_lattice_generate(N, n, seed, outputs=("digest",))
    s_bench, _ = R.rosen_lattice_generate(N, n, seed)                  # the summary-only launch bench.py times
    for key in s_bench:
        if not key.startswith("digest"):
            assert s_bench[key] == s[key], key                         # same virtual blocks: bit-identical sums
    o, _ = oracle_population("lattice", N, n, seed)
    for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
        assert s[key] == o[key], (N, key, s[key], o[key])
    for key in SUM_KEYS + ("mean_ree2", "mean_rg2", "ln_mean_W"):
        assert math.isclose(s[key], o[key], rel_tol=rel), (N, key, s[key], o[key])
    assert s["n_chains"] == n == o["n_chains"]
    compared(n, n_chains)
    return n


def check_realspace(R, w, n_chains, conf_prefix=0):
    kw = dict(k=w.k_trials, b=w.bond_len, sigma=w.sigma)
    n = affordable("realspace", w.N, n_chains, w.seed, **kw)
    s, t = R.rosen_realspace_generate(w.N, n, w.k_trials, w.bond_len, w.sigma, w.seed, outputs=("digest",))
    o, arr = oracle_population("realspace", w.N, n, w.seed, want=("digest",), **kw)
    dg_o = arr["digest"]
    dg = t["digest"].cpu().numpy().view(np.uint64)
    flips = float((dg != dg_o).mean())
    print(f"[fullpop] {w.name}: {n} chains, flip fraction {flips:.3e}")
    assert flips < 1e-4
    assert flips == 0.0            # both sides run the same IEEE operations
    for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
        assert s[key] == o[key], (key, s[key], o[key])
    for key in SUM_KEYS + ("mean_ree2", "mean_rg2", "ln_mean_W"):
        assert math.isclose(s[key], o[key], rel_tol=1e-6), (key, s[key], o[key])
    if conf_prefix:
        _, tc = R.rosen_realspace_generate(w.N, conf_prefix, w.k_trials, w.bond_len, w.sigma, w.seed, outputs=("conf", "lnW"))
        _, oc = oracle_population("realspace", w.N, conf_prefix, w.seed, want=("conf", "lnW"), **kw)
        assert np.array_equal(tc["conf"].cpu().numpy().view(np.uint32), oc["conf"].view(np.uint32))     # identical bits
        lw = tc["lnW"].cpu().numpy()
        dead = np.isneginf(oc["lnW"])
        assert np.array_equal(np.isneginf(lw), dead) and np.allclose(lw[~dead], oc["lnW"][~dead], rtol=1e-13, atol=0)
    assert s["n_chains"] == n == len(dg_o)
    compared(n, n_chains)
    return n


def test_config2_whole_population(R):
    """BASELINE config 2: all 2^24 chains of lattice N = 64, seed 7."""
    w = workloads.CONFIG_2
    check_lattice(R, w.N, w.n_chains, w.seed)


def test_config1_whole_population(R):
    w = workloads.CONFIG_1
    check_lattice(R, w.N, w.n_chains, w.seed)


@pytest.mark.parametrize("N", workloads.CONFIG_4_N)
def test_config4_whole_population(R, N):
    """BASELINE config 4 (seed 11): all 2^24 chains for N <= 128 (N = 128: 8-bit scan, step-order lnW) and the first 2^22 of
    N = 256 (hash-map kernel; the oracle's O(N^2) scan needs ~80 s for them on 16 cores)."""
    n_chains = 1 << 24 if N <= 128 else 1 << 22
    assert check_lattice(R, N, n_chains, 11) == n_chains or ALLOW_CUT


def test_config3_whole_population(R):
    """BASELINE config 3: all 2^22 real-space chains, every per-chain digest compared."""
    w = workloads.CONFIG_3
    assert check_realspace(R, w, w.n_chains) == w.n_chains or ALLOW_CUT


def test_config5_prefix_population(R):
    """BASELINE config 5 (N = 256, k = 64: 12 ms per chain on one host core): the first 2^16 chains, digests one by one --
    zero flips in 65536 chains bounds the flip rate at 4.6e-5 (95 %), below north_star's 1e-4 bar, which a 2^13 prefix
    could not resolve -- and the conformation bits of its first 2^12 chains through the dump variant."""
    assert check_realspace(R, workloads.CONFIG_5, 1 << 16, conf_prefix=1 << 12) == 1 << 16 or ALLOW_CUT


@pytest.mark.parametrize("w", workloads.MODELS, ids=lambda w: w.name)
def test_model_and_perm_bench_workloads_whole_population(R, w):
    """The four model / PERM workloads bench.py times, all 2^20 chains / tours: per-chain digest
    (every growth, enrichment and pruning decision), alive flag and attempted steps exact; lnW within 1e-12."""
    n = w.n_chains
    outs = ("digest", "alive", "lnW")
    if w.perm is not None:
        lo, hi, ref = workloads.perm_thresholds(w.N, *w.perm)
        s, t = R.rosen_lattice_perm(w.N, n, w.seed, lo, hi, ref, outputs=outs)
    elif w.kind == "lattice":
        s, t = R.rosen_lattice_generate_model(w.N, n, w.seed, z=w.z, beta_eps=w.beta_eps, outputs=outs)
    else:
        s, t = R.rosen_realspace_generate_model(w.N, n, w.k_trials, w.bond_len, w.sigma, w.lam, w.beta_eps, w.seed, outputs=outs)
    totals, arr = oracle_workload_arrays(w, n, want=outs)
    dg = t["digest"].cpu().numpy().view(np.uint64)
    assert len(dg) == n == len(arr["digest"]) == s["n_chains"]
    assert np.array_equal(dg, arr["digest"]), f"{int((dg != arr['digest']).sum())} of {n} digests differ"
    assert np.array_equal(t["alive"].cpu().numpy(), arr["alive"])
    for key in ("n_dead", "n_steps_attempted"):
        assert s[key] == totals[key], (key, s[key], totals[key])
    lw, lo_ = t["lnW"].cpu().numpy(), arr["lnW"]
    fin = np.isfinite(lo_)
    assert np.array_equal(np.isfinite(lw), fin) and np.allclose(lw[fin], lo_[fin], rtol=1e-12, atol=1e-12)
    compared(n, w.n_chains)

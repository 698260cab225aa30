"""Test helper: the unchanged single-thread oracle over a whole population, called on disjoint chain-id
ranges from a thread pool (ctypes releases the GIL during the call) and merged on the host.

Per-chain results are pure functions of (seed, chain id, parameters), so the union of the
ranges is the population; the integer fields merge exactly (sum / XOR), the fp64 sums with math.fsum.
Test infrastructure only (imports oracle/).
"""
from __future__ import annotations

import math
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

import oracle

INT_KEYS = ("n_chains", "n_dead", "n_steps_attempted")
SUM_KEYS = ("sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2")


def host_threads() -> int:
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def oracle_population(kind: str, N: int, n_chains: int, seed: int, k=None, b=None, sigma=None, chain_offset: int = 0,
                      want=(), ranges_per_thread: int = 8):
    """Returns (merged summary dict, {name: per-chain array} for the names in `want`). The ranges share the fixed shift L of short chains
    (lattice N <= 512, real space N <= 2048: DESIGN.md 3.4), which is asserted."""
    threads = host_threads()
    n_ranges = max(1, min(n_chains, threads * ranges_per_thread))
    bounds = [chain_offset + (n_chains * i) // n_ranges for i in range(n_ranges + 1)]
    outputs = tuple(want)

    def one(i):
        lo, cnt = bounds[i], bounds[i + 1] - bounds[i]
        if kind == "lattice":
            return oracle.lattice_generate(N, cnt, seed, chain_offset=lo, outputs=outputs)
        return oracle.realspace_generate(N, cnt, k, b, sigma, seed, chain_offset=lo, outputs=outputs)

    with ThreadPoolExecutor(max_workers=threads) as ex:
        parts = list(ex.map(one, range(n_ranges)))
    L = parts[0].summary["ln_shift"]
    assert all(p.summary["ln_shift"] == L for p in parts)
    m = {"ln_shift": L, "digest_xor": 0, "digest_sum": 0}
    for key in INT_KEYS:
        m[key] = sum(p.summary[key] for p in parts)
    for key in SUM_KEYS:
        m[key] = math.fsum(p.summary[key] for p in parts)
    for p in parts:
        m["digest_xor"] ^= p.summary["digest_xor"]
        m["digest_sum"] = (m["digest_sum"] + p.summary["digest_sum"]) & (2 ** 64 - 1)
    m["mean_ree2"] = m["sum_w_ree2"] / m["sum_w"]
    m["mean_rg2"] = m["sum_w_rg2"] / m["sum_w"]
    m["attrition"] = m["n_dead"] / m["n_chains"]
    m["ln_mean_W"] = L + math.log(m["sum_w"] / m["n_chains"])
    arrays = {name: np.concatenate([getattr(p, name) for p in parts]) for name in outputs}
    return m, arrays


def oracle_workload_arrays(w, n_chains: int, want=("digest",), ranges_per_thread: int = 8):
    """Per-chain arrays (and the exact integer totals) of a model / PERM workload (paper_1704_04381_b200.workloads.Workload
    with beta_eps or perm set) over chain / tour ids 0..n_chains-1. These calls shift their sums by the largest lnW of the
    CALL, so sub-range summaries do not merge by addition: whole populations are compared chain by chain instead."""
    from paper_1704_04381_b200 import workloads
    threads = host_threads()
    n_ranges = max(1, min(n_chains, threads * ranges_per_thread))
    bounds = [(n_chains * i) // n_ranges for i in range(n_ranges + 1)]
    outputs = tuple(want)
    if w.perm is not None:
        lo_thr, hi_thr, ref = workloads.perm_thresholds(w.N, *w.perm)

    def one(i):
        lo, cnt = bounds[i], bounds[i + 1] - bounds[i]
        if w.perm is not None:
            return oracle.lattice_perm(w.N, cnt, w.seed, lo_thr, hi_thr, ref, tour_offset=lo, outputs=outputs)
        if w.kind == "lattice":
            return oracle.lattice_model_generate(w.N, cnt, w.seed, z=w.z, beta_eps=w.beta_eps, chain_offset=lo, outputs=outputs)
        return oracle.realspace_model_generate(w.N, cnt, w.k_trials, w.bond_len, w.sigma, w.lam, w.beta_eps, w.seed,
                                               chain_offset=lo, outputs=outputs)

    with ThreadPoolExecutor(max_workers=threads) as ex:
        parts = list(ex.map(one, range(n_ranges)))
    totals = {key: sum(p.summary[key] for p in parts) for key in INT_KEYS}
    arrays = {name: np.concatenate([getattr(p, name) for p in parts]) for name in outputs}
    return totals, arrays

"""The synthetic workloads of BASELINE.json `configs` -- parameters only, no arithmetic of the method.

The path has no input arrays: a workload is (N, n_chains, seed, ...) and every random number is
drawn inside the path from the counter-based generator keyed by (seed, chain id, step). This
module is the single "input generator" shared by tests, bench.py, the CUDA binding callers and the
oracle callers; it imports neither of them.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional, Tuple


@dataclass(frozen=True)
class Workload:
    name: str
    kind: str                 # "lattice" | "realspace"
    N: int
    n_chains: int
    seed: int
    k_trials: Optional[int] = None
    bond_len: Optional[float] = None
    sigma: Optional[float] = None
    dump: bool = False        # full per-chain conformation output (config 5)
    z: int = 6                # lattice trial set (model calls: 6 or 26)
    beta_eps: Optional[float] = None   # contact / well depth in kT: not None selects the model call
    lam: Optional[float] = None        # real-space well range in units of sigma
    perm: Optional[Tuple[float, float]] = None   # PERM: thresholds (lo, hi) x the asymptotic c_n

    def monomer_steps_nominal(self) -> int:
        return self.n_chains * (self.N - 1)


# BASELINE.json configs[0..4]; config 3 has no seed in BASELINE.json: seed = 3.
CONFIG_1 = Workload("lattice_N16_2p16", "lattice", 16, 1 << 16, 1)
CONFIG_2 = Workload("lattice_N64_2p24", "lattice", 64, 1 << 24, 7)
CONFIG_3 = Workload("realspace_N64_k16_2p22", "realspace", 64, 1 << 22, 3, 16, 1.0, 1.0)
CONFIG_4_N: Tuple[int, ...] = (8, 16, 32, 64, 128, 256)
CONFIG_4 = tuple(Workload(f"lattice_sweep_N{N}_2p24", "lattice", N, 1 << 24, 11) for N in CONFIG_4_N)
CONFIG_5 = Workload("realspace_N256_k64_2p20_dump", "realspace", 256, 1 << 20, 13, 64, 1.0, 0.8, dump=True)

# Beyond BASELINE.json: the long lattice chains of the paper's Table 1,
# N = 1024 / 2048 of the shared-memory rows and N = 10000, the longest "global-memory version" row.
LONG_LATTICE = (Workload("lattice_long_N1024_2p20", "lattice", 1024, 1 << 20, 17),
                Workload("lattice_long_N2048_2p19", "lattice", 2048, 1 << 19, 17),
                Workload("lattice_long_N10000_2p17", "lattice", 10000, 1 << 17, 17),      # 1.7 chains per resident thread: tail-dominated
                Workload("lattice_long_N10000_2p20", "lattice", 10000, 1 << 20, 17))

# ... and of Table 2; the paper does not state its trial set: config 3's (k = 16, b = sigma = 1,
# where 96 % of the chains die before N = 4096) and config 5's (k = 64, sigma = 0.8, where nearly all reach N = 10000).
LONG_REALSPACE = (Workload("realspace_long_N4096_k16_2p16", "realspace", 4096, 1 << 16, 17, 16, 1.0, 1.0),
                  Workload("realspace_long_N10000_k64_2p14", "realspace", 10000, 1 << 14, 17, 64, 1.0, 0.8))

# other trial sets / Boltzmann-weighted trials, PERM (n_chains = tours there)
MODELS = (Workload("lattice_z26_N64_2p20", "lattice", 64, 1 << 20, 19, z=26, beta_eps=0.0),
          Workload("lattice_z6_contact0.3_N64_2p20", "lattice", 64, 1 << 20, 19, z=6, beta_eps=0.3),
          Workload("realspace_well1.5_0.4_N64_k16_2p20", "realspace", 64, 1 << 20, 19, 16, 1.0, 1.0, beta_eps=0.4, lam=1.5),
          Workload("lattice_perm_N256_2p20", "lattice", 256, 1 << 20, 19, perm=(0.5, 2.0)))

CONFIGS = {w.name: w for w in (CONFIG_1, CONFIG_2, CONFIG_3, *CONFIG_4, CONFIG_5, *LONG_LATTICE, *LONG_REALSPACE, *MODELS)}


def perm_thresholds(N: int, lo: float, hi: float):
    """ln_lo, ln_hi [N+1] and ln_ref for PERM: (lo, hi) x the asymptotic form c_n ~ 1.21 mu^n n^(gamma-1), mu = 4.684,
    gamma = 1.157 (control parameters only: the PERM estimate is unbiased for any thresholds)."""
    import math
    ln_c = [0.0, 0.0] + [math.log(1.21) + (n - 1) * math.log(4.684) + 0.157 * math.log(n - 1) for n in range(2, N + 1)]
    return [v + math.log(lo) for v in ln_c], [v + math.log(hi) for v in ln_c], ln_c[N]


def shard(n_chains: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous chain-id range [offset, offset+count) of `rank` among `world` ranks (balanced)."""
    base, rem = divmod(n_chains, world)
    count = base + (1 if rank < rem else 0)
    offset = rank * base + min(rank, rem)
    return offset, count

"""CPU oracle for the Rosenbluth chain-generation hot path -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package. It is a ctypes front-end over
``oracle/librosen_oracle.so`` (plain single-threaded C++, built by ``oracle/build.py``) and
shares nothing with ``paper_1704_04381_b200`` -- neither imports the other.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

from .build import build as _build

_LIB: Optional[C.CDLL] = None


class _Summary(C.Structure):
    _fields_ = [
        ("n_chains", C.c_uint64), ("n_dead", C.c_uint64), ("n_steps_attempted", C.c_uint64),
        ("ln_shift", C.c_double),
        ("sum_w", C.c_double), ("sum_w_ree2", C.c_double), ("sum_w_rg2", C.c_double), ("sum_w2", C.c_double),
        ("mean_ree2", C.c_double), ("mean_rg2", C.c_double), ("attrition", C.c_double), ("ln_mean_W", C.c_double),
        ("digest_xor", C.c_uint64), ("digest_sum", C.c_uint64),
    ]


class _Outputs(C.Structure):
    _fields_ = [
        ("lnW", C.c_void_p), ("alive", C.c_void_p), ("m_seq", C.c_void_p), ("digest", C.c_void_p),
        ("conf", C.c_void_p), ("ree2", C.c_void_p), ("rg2", C.c_void_p),
    ]


def lib() -> C.CDLL:
    global _LIB
    if _LIB is None:
        path = _build()
        L = C.CDLL(path)
        L.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.oracle_philox4x32_10.restype = None
        L.oracle_lattice_free_dirs.argtypes = [C.POINTER(C.c_int32), C.c_int32, C.POINTER(C.c_int32)]
        L.oracle_lattice_free_dirs.restype = C.c_int32
        L.oracle_direction.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(C.c_float)]
        L.oracle_direction.restype = None
        L.oracle_lattice_generate.argtypes = [C.c_int32, C.c_uint64, C.c_uint64, C.c_uint64,
                                              C.POINTER(_Outputs), C.POINTER(_Summary)]
        L.oracle_lattice_generate.restype = C.c_int
        L.oracle_realspace_generate.argtypes = [C.c_int32, C.c_uint64, C.c_int32, C.c_float, C.c_float,
                                                C.c_uint64, C.c_uint64, C.POINTER(_Outputs), C.POINTER(_Summary)]
        L.oracle_realspace_generate.restype = C.c_int
        L.oracle_saw_enumerate.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64),
                                           C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.oracle_saw_enumerate.restype = C.c_int
        L.oracle_model_table.argtypes = [C.c_double, C.POINTER(C.c_uint64)]
        L.oracle_model_table.restype = None
        L.oracle_scaled_target.argtypes = [C.c_uint32, C.c_uint64]
        L.oracle_scaled_target.restype = C.c_uint64
        L.oracle_lattice_model_step.argtypes = [C.POINTER(C.c_int32), C.c_int32, C.c_int32, C.POINTER(C.c_uint64),
                                                C.POINTER(C.c_uint64)]
        L.oracle_lattice_model_step.restype = C.c_int32
        L.oracle_lattice_model_generate.argtypes = [C.c_int32, C.c_uint64, C.c_uint64, C.c_uint64, C.c_int32, C.c_double,
                                                    C.POINTER(_Outputs), C.POINTER(_Summary)]
        L.oracle_lattice_model_generate.restype = C.c_int
        L.oracle_realspace_model_generate.argtypes = [C.c_int32, C.c_uint64, C.c_int32, C.c_float, C.c_float, C.c_float,
                                                      C.c_double, C.c_uint64, C.c_uint64, C.POINTER(_Outputs),
                                                      C.POINTER(_Summary)]
        L.oracle_realspace_model_generate.restype = C.c_int
        L.oracle_saw_enumerate_model.argtypes = [C.c_int32, C.c_int32, C.c_double, C.POINTER(C.c_double)]
        L.oracle_saw_enumerate_model.restype = C.c_int
        L.oracle_lattice_perm.argtypes = [C.c_int32, C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_double),
                                          C.POINTER(C.c_double), C.c_double, C.c_uint64, C.POINTER(_Outputs), C.POINTER(_Summary)]
        L.oracle_lattice_perm.restype = C.c_int
        _LIB = L
    return _LIB


@dataclass
class Result:
    """Summary (dict of python scalars) and the requested per-chain numpy arrays."""
    summary: dict
    lnW: Optional[np.ndarray] = None
    alive: Optional[np.ndarray] = None
    m_seq: Optional[np.ndarray] = None
    digest: Optional[np.ndarray] = None
    conf: Optional[np.ndarray] = None
    ree2: Optional[np.ndarray] = None
    rg2: Optional[np.ndarray] = None


def _alloc(n_chains: int, N: int, conf_dtype, want: set):
    arrs = {}
    if "lnW" in want: arrs["lnW"] = np.empty(n_chains, np.float64)
    if "alive" in want: arrs["alive"] = np.empty(n_chains, np.uint8)
    if "m_seq" in want: arrs["m_seq"] = np.empty((n_chains, N - 1), np.uint8)
    if "digest" in want: arrs["digest"] = np.empty(n_chains, np.uint64)
    if "conf" in want: arrs["conf"] = np.empty((n_chains, N, 3), conf_dtype)
    if "ree2" in want: arrs["ree2"] = np.empty(n_chains, np.float64)
    if "rg2" in want: arrs["rg2"] = np.empty(n_chains, np.float64)
    out = _Outputs(*[arrs[k].ctypes.data if k in arrs else None
                     for k in ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")])
    return arrs, out


ALL = ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")


def _summary_dict(s: _Summary) -> dict:
    return {name: getattr(s, name) for name, _ in _Summary._fields_}


def lattice_generate(N: int, n_chains: int, seed: int, chain_offset: int = 0, outputs=ALL) -> Result:
    arrs, out = _alloc(n_chains, N, np.int32, set(outputs))
    s = _Summary()
    rc = lib().oracle_lattice_generate(N, n_chains, seed, chain_offset, C.byref(out), C.byref(s))
    if rc != 0:
        raise ValueError(f"oracle_lattice_generate: invalid arguments (rc={rc})")
    return Result(summary=_summary_dict(s), **arrs)


def realspace_generate(N: int, n_chains: int, k_trials: int, bond_len: float, sigma: float, seed: int,
                       chain_offset: int = 0, outputs=ALL) -> Result:
    arrs, out = _alloc(n_chains, N, np.float32, set(outputs))
    s = _Summary()
    rc = lib().oracle_realspace_generate(N, n_chains, k_trials, bond_len, sigma, seed, chain_offset,
                                         C.byref(out), C.byref(s))
    if rc != 0:
        raise ValueError(f"oracle_realspace_generate: invalid arguments (rc={rc})")
    return Result(summary=_summary_dict(s), **arrs)


def lattice_model_generate(N: int, n_chains: int, seed: int, z: int = 6, beta_eps: float = 0.0, chain_offset: int = 0,
                           outputs=ALL) -> Result:
    """Lattice chains with the z = 6 / 26 trial set and contact energy -eps per non-bonded neighbour pair
    (Boltzmann-weighted trials)."""
    arrs, out = _alloc(n_chains, N, np.int32, set(outputs))
    s = _Summary()
    rc = lib().oracle_lattice_model_generate(N, n_chains, seed, chain_offset, z, beta_eps, C.byref(out), C.byref(s))
    if rc != 0:
        raise ValueError(f"oracle_lattice_model_generate: invalid arguments (rc={rc})")
    return Result(summary=_summary_dict(s), **arrs)


def realspace_model_generate(N: int, n_chains: int, k_trials: int, bond_len: float, sigma: float, lam: float,
                             beta_eps: float, seed: int, chain_offset: int = 0, outputs=ALL) -> Result:
    """Real-space chains with a square-well attraction of range lam * sigma and depth eps."""
    arrs, out = _alloc(n_chains, N, np.float32, set(outputs))
    s = _Summary()
    rc = lib().oracle_realspace_model_generate(N, n_chains, k_trials, bond_len, sigma, lam, beta_eps, seed, chain_offset,
                                               C.byref(out), C.byref(s))
    if rc != 0:
        raise ValueError(f"oracle_realspace_model_generate: invalid arguments (rc={rc})")
    return Result(summary=_summary_dict(s), **arrs)


def model_table(beta_eps: float) -> list:
    q = (C.c_uint64 * 32)()
    lib().oracle_model_table(beta_eps, q)
    return [int(v) for v in q]


def scaled_target(u: int, W: int) -> int:
    """floor(u W / 2^32) as the model oracles compute it (the threshold of the Boltzmann-proportional choice)."""
    return int(lib().oracle_scaled_target(u, W))


def lattice_model_step(r: np.ndarray, z: int, beta_eps: float) -> list:
    """Per-trial fixed-point weights (0 = occupied) for the next monomer of walk r [s][3]."""
    r = np.ascontiguousarray(r, dtype=np.int32)
    q = (C.c_uint64 * 32)(*model_table(beta_eps))
    w = (C.c_uint64 * 26)()
    lib().oracle_lattice_model_step(r.ctypes.data_as(C.POINTER(C.c_int32)), r.shape[0], z, q, w)
    return [int(w[d]) for d in range(z)]


def saw_enumerate_model(n: int, z: int, beta_eps: float) -> dict:
    out = (C.c_double * 5)()
    rc = lib().oracle_saw_enumerate_model(n, z, beta_eps, out)
    if rc != 0:
        raise RuntimeError(f"oracle_saw_enumerate_model rc={rc}")
    return dict(zip(("count", "sum_boltz", "sum_boltz_ree2", "sum_quant", "sum_prob"), [float(v) for v in out]))


def lattice_perm(N: int, n_tours: int, seed: int, ln_lo, ln_hi, ln_ref: float, max_nodes: int = 1 << 20, tour_offset: int = 0,
                 outputs=("lnW", "alive", "digest", "ree2", "rg2")) -> Result:
    """PERM tours on the cubic lattice with caller-given thresholds ln_lo / ln_hi [N+1] (index = number of monomers,
    entries 2..N-1 used); per-tour results in the per-chain fields (see rosen_oracle.cpp)."""
    lo = np.ascontiguousarray(ln_lo, dtype=np.float64); hi = np.ascontiguousarray(ln_hi, dtype=np.float64)
    assert lo.shape == (N + 1,) and hi.shape == (N + 1,)
    arrs, out = _alloc(n_tours, N, np.int32, set(outputs) - {"conf", "m_seq"})
    s = _Summary()
    rc = lib().oracle_lattice_perm(N, n_tours, seed, tour_offset, lo.ctypes.data_as(C.POINTER(C.c_double)),
                                   hi.ctypes.data_as(C.POINTER(C.c_double)), ln_ref, max_nodes, C.byref(out), C.byref(s))
    if rc != 0:
        raise ValueError(f"oracle_lattice_perm: invalid arguments (rc={rc})")
    return Result(summary=_summary_dict(s), **arrs)


def philox4x32_10(ctr, key) -> tuple:
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def lattice_free_dirs(r: np.ndarray) -> list:
    """Free trial directions (indices into +x,-x,+y,-y,+z,-z) for the next monomer of walk r [s][3]."""
    r = np.ascontiguousarray(r, dtype=np.int32)
    fd = (C.c_int32 * 6)()
    m = lib().oracle_lattice_free_dirs(r.ctypes.data_as(C.POINTER(C.c_int32)), r.shape[0], fd)
    return [int(fd[i]) for i in range(m)]


def direction(wz: int, wphi: int) -> np.ndarray:
    u = (C.c_float * 3)()
    lib().oracle_direction(wz & 0xFFFFFFFF, wphi & 0xFFFFFFFF, u)
    return np.array([u[0], u[1], u[2]], dtype=np.float32)


def saw_enumerate(n: int, fix_first: bool = False) -> dict:
    """Brute-force enumeration of n-step cubic-lattice SAWs; see saw_enum.cpp.

    Returns count, sum_ree2, sum_n2rg2 (integers, already multiplied by 6 when fix_first) and
    ``hist``: dict {(a, b, c): number of walks with W = 2^a 3^b 5^c}.
    """
    hist = np.zeros((2 * n + 1, n + 1, n + 1), dtype=np.uint64)
    cnt, s1, s2 = C.c_uint64(), C.c_uint64(), C.c_uint64()
    rc = lib().oracle_saw_enumerate(n, int(fix_first), C.byref(cnt), C.byref(s1), C.byref(s2),
                                    hist.ctypes.data_as(C.POINTER(C.c_uint64)))
    if rc != 0:
        raise RuntimeError(f"oracle_saw_enumerate rc={rc}")
    mult = 6 if fix_first else 1
    h = {tuple(int(i) for i in idx): int(hist[tuple(idx)]) * mult for idx in np.argwhere(hist)}
    return {"count": cnt.value * mult, "sum_ree2": s1.value * mult, "sum_n2rg2": s2.value * mult, "hist": h}


def fit_exponents(N, mean_ree2, ln_mean_W, use_steps: bool = True) -> dict:
    """Scaling analysis of a length sweep, PAPER.md:342-367 (sec. 4.1): Eq. 4 <R_N^2> = a N^(2 nu) and
    Eq. 7 ln Z_N = c + N ln mu + (gamma - 1) ln N with Z_N = <W_N> (Eq. 6), each as the plain linear
    least-squares problem it states, solved by numpy.linalg.lstsq. x = N - 1 when use_steps (reading A14)."""
    x = np.asarray(N, dtype=np.float64) - (1.0 if use_steps else 0.0)
    lx = np.log(x)
    A1 = np.stack([np.ones_like(lx), lx], axis=1)
    (ln_a, slope), *_ = np.linalg.lstsq(A1, np.log(np.asarray(mean_ree2, dtype=np.float64)), rcond=None)
    out = {"nu": 0.5 * slope, "ln_a": ln_a, "mu": float("nan"), "gamma": float("nan"), "c": float("nan")}
    if len(x) >= 3:
        A2 = np.stack([np.ones_like(lx), x, lx], axis=1)
        (c, ln_mu, gm1), *_ = np.linalg.lstsq(A2, np.asarray(ln_mean_W, dtype=np.float64), rcond=None)
        out.update(mu=float(np.exp(ln_mu)), gamma=float(gm1 + 1.0), c=float(c))
    return out

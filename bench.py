#!/usr/bin/env python
"""bench.py -- one JSON line for the Rosenbluth chain-generation hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

A "step" is one pass of the whole hot path (L0-L5 + E1, or R0-R5 + E1 [+ D1]) over one
batch of the workload, i.e. one rosen_*_generate call. Default workload = BASELINE.json configs[1]
(cubic lattice, N = 64, 2^24 chains, seed 7), the configuration the metric is quoted on.

  value      chains/s, device-timed (CUDA events on the launching stream), outputs resident in HBM
             (rosen_*_generate_async: generation kernel + second reduction pass, no host sync)
  e2e        the same metric through the synchronous C-ABI call with HOST buffers (summary struct, and for
             the dump workload the conformations) -- device->host copies inside the timed region
  roofline   bound "alu": algorithmic warp-instructions / live kernel time vs issue-slot peak
  cpu_baseline  the oracle as it stands on all host cores (and on one), on a bounded sample of the same workload

N > 1 (torchrun): chains are independent, so every rank generates its own n_chains with
chain_offset = rank * n_chains (weak scaling, no data-path collective); summaries are merged on
the host after the timed region (rosen_summary_merge).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1704_04381_b200 import workloads  # noqa: E402  (parameters only)

DEFAULT_WORKLOAD = workloads.CONFIG_2.name
METRIC = "chains/sec and monomer-steps/sec at N=64 (1 B200); % SM issue-slot peak"


# ------------------------------------------------------------------------------------------------
# algorithmic work model -- thread-instructions the METHOD needs per chain
# ------------------------------------------------------------------------------------------------
def lattice_site_tests(N: int) -> int:
    """Site tests per chain after the exact bipartite + back-site reduction: sum_s max(0, floor(s/2) - 1)."""
    return sum(max(0, s // 2 - 1) for s in range(1, N))


HASH_INSTR_PER_STEP = 123.5     # hash-map lattice kernel (N >= 193), per attempted step; see run_product


def algorithmic_thread_instr(w: workloads.Workload) -> float:
    if w.kind == "lattice":
        # 6 equality tests per site test + one Philox block (~70 instr) per 4 steps + ~20 per step for
        # count / weight / choose / place / observables
        return 6.0 * lattice_site_tests(w.N) + 70.0 * ((w.N + 3) // 4) + 20.0 * (w.N - 1)
    # real space after the exact candidate reduction (DESIGN.md 5.2 / 6): (N-1)(N-2)/2 prefilter tests and
    # k * c pair tests per step with c = 3.2 candidates on average, 7 instr each, + k/2 Philox
    # blocks (35 per trial) and k direction evaluations (45) per step + ~30 per step
    k, N = w.k_trials, w.N
    return 7.0 * (N - 1) * (N - 2) / 2.0 + (N - 1) * (7.0 * 3.2 * k + 35.0 * k + 45.0 * k + 30.0)


PROFILE_OF = {   # committed ncu summary (profiles/) of the dominant kernel of each workload
    "lattice_N16_2p16": "r02_lattice_cfg1.md", "lattice_N64_2p24": "r02_lattice_cfg2.md",
    "realspace_N64_k16_2p22": "r02_realspace_cfg3.md", "realspace_N256_k64_2p20_dump": "r02_realspace_cfg5.md",
    "lattice_sweep_N128_2p24": "r02_lattice_sweep_N128.md", "lattice_sweep_N256_2p24": "r02_lattice_sweep_N256.md",
    "lattice_long_N1024_2p20": "r02_lattice_long_N1024.md", "lattice_long_N2048_2p19": "r02_lattice_long_N2048.md",
    "lattice_long_N10000_2p17": "r02_lattice_long_N10000.md", "realspace_long_N4096_k16_2p16": "r02_realspace_long_N4096.md",
    "realspace_long_N10000_k64_2p14": "r02_realspace_long_N10000.md",
    "lattice_z6_contact0.3_N64_2p20": "r03_lattice_model_z6.md", "lattice_z26_N64_2p20": "r03_lattice_model_z26.md",
    "realspace_well1.5_0.4_N64_k16_2p20": "r03_realspace_well.md", "lattice_perm_N256_2p20": "r03_lattice_perm.md",
}


def profile_metrics(w: workloads.Workload) -> dict:
    """Per-launch metrics of the dominant kernel from the committed ncu summary of this workload (profiles/): DRAM traffic,
    warp-instructions executed, threads per instruction, issue-active %. Empty if no capture is committed."""
    name = PROFILE_OF.get(w.name)
    path = os.path.join(ROOT, "profiles", name) if name else None
    if not path or not os.path.exists(path):
        return {}
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    out = {"file": "profiles/" + name}
    traffic = None
    for line in open(path):
        cells = [c.strip() for c in line.split("|")]
        if len(cells) < 4:
            continue
        try:
            if cells[1] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                traffic = (traffic or 0.0) + float(cells[3]) * mult.get(cells[2], 1.0)
            elif cells[1] == "smsp__inst_executed.sum":
                out["warp_inst_executed"] = float(cells[3])
            elif cells[1] == "smsp__thread_inst_executed_per_inst_executed.ratio":
                out["active_lane_ratio"] = float(cells[3])
            elif cells[1] == "smsp__issue_active.avg.pct_of_peak_sustained_active":
                out["issue_active_pct"] = float(cells[3])
        except ValueError:
            continue
    out["traffic"] = traffic
    return out


def load_measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ------------------------------------------------------------------------------------------------
# clock sampling during the timed region (B200_PROFILING.md "clocks line")
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [ln for (t, ln) in self.lines if t0 <= t <= t1 + 0.1] or [ln for (_, ln) in self.lines]
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in rows:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# the two legs of the product path
# ------------------------------------------------------------------------------------------------
def make_calls(R, torch, w: workloads.Workload, offset: int, stream):
    """Return (enqueue(summary_device_or_None), sync_call(), d2h_bytes) for workload w."""
    dump = {}
    host = {}
    if w.dump:   # config 5: conformations + lnW written to HBM (D1)
        ctype = torch.int32 if w.kind == "lattice" else torch.float32
        dump = {"conf": torch.empty((w.n_chains, w.N, 3), dtype=ctype, device="cuda"),
                "lnW": torch.empty((w.n_chains,), dtype=torch.float64, device="cuda")}
    d2h = R.SUMMARY_BYTES + sum(t.numel() * t.element_size() for t in dump.values())

    if w.perm is not None or w.beta_eps is not None:
        # model / PERM calls have no _async twin: the device-timed leg enqueues the call without a
        # host summary (no synchronisation), the end-to-end leg takes the summary
        if w.perm is not None:
            lo, hi, ref = workloads.perm_thresholds(w.N, *w.perm)

            def call(summary):
                return R.rosen_lattice_perm(w.N, w.n_chains, w.seed, lo, hi, ref, tour_offset=offset, stream=stream, summary=summary)[0]
        elif w.kind == "lattice":
            def call(summary):
                return R.rosen_lattice_generate_model(w.N, w.n_chains, w.seed, z=w.z, beta_eps=w.beta_eps, chain_offset=offset,
                                                      stream=stream, summary=summary)[0]
        else:
            def call(summary):
                return R.rosen_realspace_generate_model(w.N, w.n_chains, w.k_trials, w.bond_len, w.sigma, w.lam, w.beta_eps, w.seed,
                                                        chain_offset=offset, stream=stream, summary=summary)[0]
        return (lambda summary_device: call(False)), (lambda: call(True)), d2h
    if w.kind == "lattice":
        def enqueue(summary_device):
            R.rosen_lattice_generate_async(w.N, w.n_chains, w.seed, offset, outputs=dump,
                                           summary_device=summary_device, stream=stream)

        def sync_call():
            s, t = R.rosen_lattice_generate(w.N, w.n_chains, w.seed, offset, outputs=tuple(dump), stream=stream,
                                            host_outputs=True, host_buffers=host)
            return s
    else:
        def enqueue(summary_device):
            R.rosen_realspace_generate_async(w.N, w.n_chains, w.k_trials, w.bond_len, w.sigma, w.seed, offset,
                                             outputs=dump, summary_device=summary_device, stream=stream)

        def sync_call():
            s, t = R.rosen_realspace_generate(w.N, w.n_chains, w.k_trials, w.bond_len, w.sigma, w.seed, offset,
                                              outputs=tuple(dump), stream=stream, host_outputs=True, host_buffers=host)
            return s
    return enqueue, sync_call, d2h


def oracle_call(w: workloads.Workload, n_chains: int, offset: int = 0):
    import oracle  # test infrastructure; allowed here for cpu_baseline / --impl reference only
    if w.perm is not None:
        lo, hi, ref = workloads.perm_thresholds(w.N, *w.perm)
        return oracle.lattice_perm(w.N, n_chains, w.seed, lo, hi, ref, tour_offset=offset, outputs=())
    if w.beta_eps is not None and w.kind == "lattice":
        return oracle.lattice_model_generate(w.N, n_chains, w.seed, z=w.z, beta_eps=w.beta_eps, chain_offset=offset, outputs=())
    if w.beta_eps is not None:
        return oracle.realspace_model_generate(w.N, n_chains, w.k_trials, w.bond_len, w.sigma, w.lam, w.beta_eps, w.seed,
                                               chain_offset=offset, outputs=())
    if w.kind == "lattice":
        return oracle.lattice_generate(w.N, n_chains, w.seed, chain_offset=offset, outputs=())
    return oracle.realspace_generate(w.N, n_chains, w.k_trials, w.bond_len, w.sigma, w.seed, chain_offset=offset,
                                     outputs=())


def time_oracle(w: workloads.Workload, target_s: float):
    """Single-thread oracle on a chain-id prefix sized for about target_s seconds."""
    probe = 64 if w.N <= 2048 else 1                     # a long chain can cost seconds by itself
    while True:
        t0 = time.perf_counter(); oracle_call(w, probe); dt = time.perf_counter() - t0
        if dt > 0.2 or probe >= w.n_chains:
            break
        probe *= 4
    m = int(min(w.n_chains, max(probe, probe * target_s / max(dt, 1e-9))))
    t0 = time.perf_counter(); res = oracle_call(w, m); dt = time.perf_counter() - t0
    return m, dt, res.summary


def time_oracle_all_cores(w: workloads.Workload, per_thread: int, threads: int):
    """The unchanged single-thread oracle called on disjoint chain-id ranges from `threads` host threads (ctypes
    releases the GIL during the call). Returns (chains, seconds)."""
    from concurrent.futures import ThreadPoolExecutor
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(lambda i: oracle_call(w, per_thread, offset=i * per_thread), range(threads)))
    return per_thread * threads, time.perf_counter() - t0


def model_thread_instr(w: workloads.Workload):
    """(thread-instructions, "per chain" | "per attempted step") the METHOD needs for a model / PERM workload (DESIGN.md 6,
    round 3): the base models with the terms these variants add.
      lattice model   per chain: the box scan 8 per earlier monomer (3 coordinate range tests, map bit) over sum_s (s - 1)
                      monomers; per step z trials x (occupancy 2 + weight / count / cumulative selection 5, + 4 for the
                      contact popcount when beta eps > 0) + a quarter Philox block 17.5 + 30 (log, place, sums, digest)
      square well     the config-3 model with 8 instead of 7 per pair test (second compare), 3 per trial for the
                      fixed-point weight and its prefix sum, and 3.2 x ((b + lambda sigma) / (b + sigma))^3 candidates per
                      trial (the candidate sphere reaches to the well's edge)
      PERM            per node: 6 per site test over the (n - 2) / 2 monomers of the right parity, n ~ N / 2 on average over
                      the nodes of a tour (approximation: the length distribution of nodes is flat to within the
                      enrichment / pruning balance), + one Philox block 70 + 30 (count, choose, place, thresholds, stack)"""
    N, k = w.N, w.k_trials
    if w.perm is not None:
        return 6.0 * (N / 2.0 - 2.0) / 2.0 + 70.0 + 30.0, "per attempted step"
    if w.kind == "lattice":
        per_trial = 7.0 + (4.0 if (w.beta_eps or 0.0) > 0.0 else 0.0)
        return 8.0 * (N - 1) * (N - 2) / 2.0 + (N - 1) * (w.z * per_trial + 17.5 + 30.0), "per chain"
    # candidates per trial grow with the volume of the candidate sphere: radius b + lambda sigma instead of b + sigma
    cand = 3.2 * ((w.bond_len + w.lam * w.sigma) / (w.bond_len + w.sigma)) ** 3
    return 7.0 * (N - 1) * (N - 2) / 2.0 + (N - 1) * (8.0 * cand * k + 35.0 * k + 45.0 * k + 3.0 * k + 30.0), "per chain"


def alg_warp_inst(w: workloads.Workload, steps_attempted: float):
    """Algorithmic warp-instructions of one launch under the models of DESIGN.md 6, and the model in words (the same
    numbers run_product uses for the headline workload)."""
    if w.perm is not None or w.beta_eps is not None:
        per, unit = model_thread_instr(w)
        return per * (steps_attempted if unit == "per attempted step" else w.n_chains) / 32.0, f"{per:.1f} thread-instr {unit}"
    if w.kind == "lattice" and w.N >= 193:
        return HASH_INSTR_PER_STEP * steps_attempted / 32.0, f"{HASH_INSTR_PER_STEP} thread-instr per attempted step (hash-map kernel)"
    if w.kind == "realspace" and w.N >= 400:
        per = w.k_trials * (80.0 + 7.0 * 3.2) + 27 * 14.0 + 40 * 10.0 + 50.0
        return per * steps_attempted / 32.0, f"{per:.1f} thread-instr per attempted step (cell-list kernel)"
    per = algorithmic_thread_instr(w)
    return per * w.n_chains / 32.0, f"{per:.0f} thread-instr per chain"


def oracle_digests(w: workloads.Workload, n: int):
    """Per-chain digests of chain ids [0, n) from the oracle on all host cores (disjoint ranges, results concatenated)."""
    import numpy as np
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    threads = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    parts = max(1, min(n, threads * 4))
    bounds = [n * i // parts for i in range(parts + 1)]

    def one(i):
        return oracle.realspace_generate(w.N, bounds[i + 1] - bounds[i], w.k_trials, w.bond_len, w.sigma, w.seed,
                                         chain_offset=bounds[i], outputs=("digest",)).digest
    with ThreadPoolExecutor(max_workers=threads) as ex:
        return np.concatenate(list(ex.map(one, range(parts))))


def measure_brief(R, torch, w: workloads.Workload, stream, timed, peak_winst: float, hbm_gbs: float, steps: int, flip_sample: int):
    """One entry of the `configs` block: workload w timed in this process with the method of the headline leg (CUDA events
    on the launching stream, L2 flushed between steps, 3 warm-up steps), generation kernel alone, the synchronous
    host-buffer call end to end, the roofline fraction under the DESIGN.md 6 model, and for real space the flip fraction
    of the first `flip_sample` chains against the oracle and (dump workload) the store-phase bandwidth."""
    enqueue, sync_call, d2h_bytes = make_calls(R, torch, w, 0, stream)
    summary_dev = torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda")
    timed(lambda: enqueue(summary_dev), 3)
    launches, kernel_name = R.rosen_last_launch_count(), R.rosen_last_kernel_name()
    ms = timed(lambda: enqueue(summary_dev), steps)
    summary = R.summary_from_device(summary_dev)
    timed(lambda: enqueue(None), 1)
    kms = timed(lambda: enqueue(None), max(3, steps // 2))
    kernel_ms = sum(kms) / len(kms)
    sync_call()
    e0 = time.perf_counter()
    for _ in range(3):
        sync_call()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - e0) / 3 * 1e3
    ms_per_step = sum(ms) / len(ms)
    alg, model = alg_warp_inst(w, summary["n_steps_attempted"])
    entry = {
        "N": w.N, "n_chains": w.n_chains, "seed": w.seed, "k_trials": w.k_trials, "steps": steps, "warmup": 3,
        "ms_per_step": ms_per_step, "chains_per_s": w.n_chains / (ms_per_step * 1e-3),
        "monomer_steps_per_s": summary["n_steps_attempted"] / (ms_per_step * 1e-3),
        "kernel": kernel_name, "kernel_ms": kernel_ms, "gpu_launches_per_step": launches,
        "roofline": {"bound": "alu", "frac": alg / (kernel_ms * 1e-3) / peak_winst, "achieved": alg / (kernel_ms * 1e-3) / 1e9,
                     "peak": peak_winst / 1e9, "unit": "Gwarp-inst/s", "model": model},
        "e2e_ms_per_step": e2e_ms, "e2e_chains_per_s": w.n_chains / (e2e_ms * 1e-3), "d2h_bytes_per_step": d2h_bytes,
        "attrition": summary["attrition"], "mean_ree2": summary["mean_ree2"],
    }
    if w.kind == "realspace" and flip_sample:
        import numpy as np
        n = min(flip_sample, w.n_chains)
        _, tg = R.rosen_realspace_generate(w.N, n, w.k_trials, w.bond_len, w.sigma, w.seed, outputs=("digest",))
        ref = oracle_digests(w, n)
        entry["flip_fraction"] = {"value": float((tg["digest"].cpu().numpy().view(np.uint64) != ref).mean()), "chains": n, "bar": 1e-4}
    if w.dump and w.kind == "realspace":
        def gen_only():
            R.rosen_realspace_generate_async(w.N, w.n_chains, w.k_trials, w.bond_len, w.sigma, w.seed, 0, outputs=None,
                                             summary_device=None, stream=stream)
        conf = torch.empty((w.n_chains, w.N, 3), dtype=torch.float32, device="cuda")
        lnw = torch.empty((w.n_chains,), dtype=torch.float64, device="cuda")
        timed(gen_only, 1)
        t_gen, t_all = min(timed(gen_only, 3)), min(kms)
        timed(lambda: R.rosen_realspace_dump_probe(w.N, w.n_chains, conf, lnw, stream=stream), 2)
        t_probe = min(timed(lambda: R.rosen_realspace_dump_probe(w.N, w.n_chains, conf, lnw, stream=stream), 5))
        nbytes = w.n_chains * (12 * w.N + 8)
        diff = t_all - t_gen
        entry["dump_path"] = {"bytes_per_step": nbytes, "with_dump_ms": t_all, "generation_only_ms": t_gen,
                              "in_situ_store_GBps": nbytes / (diff * 1e-3) / 1e9 if diff > 0.01 * t_all else None,
                              "isolated_store_ms": t_probe, "isolated_store_GBps": nbytes / (t_probe * 1e-3) / 1e9,
                              "peak_GBps": hbm_gbs, "isolated_store_frac": nbytes / (t_probe * 1e-3) / 1e9 / hbm_gbs}
        del conf, lnw
    return entry


def run_reference(args, w, rank):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    warmup, steps = max(args.warmup, 1), args.steps
    m0, dt0, _ = time_oracle(w, 1.0)
    budget = 120.0 / (steps + warmup)                    # whole run within a few minutes
    m = int(max(16 if w.N <= 2048 else 1, min(w.n_chains, m0 / dt0 * min(budget, 2.0))))
    for _ in range(warmup):
        oracle_call(w, m)
    t0 = time.perf_counter()
    n_steps = 0
    for i in range(steps):
        n_steps += oracle_call(w, m, offset=i * m).summary["n_steps_attempted"]
    dt = time.perf_counter() - t0
    v = steps * m / dt
    sample = f"{m} chains per step (chain-id ranges [i*{m}, (i+1)*{m})) of {w.name}, single thread"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "chains/s", "n_gpus": args.gpus, "steps": steps,
        "warmup": warmup, "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32+f64" if w.kind == "lattice" else "f32+f64", "data": "synthetic",
        "config": {"workload": w.name, "kind": w.kind, "N": w.N, "chains_per_step": m, "seed": w.seed},
        "monomer_steps_per_s": n_steps / dt,
        "cpu_baseline": {"value": v, "unit": "chains/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "chains/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_product(args, w, rank, world, local_rank):
    import torch
    import paper_1704_04381_b200 as R

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    R.load_library()                                       # fails loudly if librosen.so is missing
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    warmup, steps = max(args.warmup, 3), args.steps
    stream = torch.cuda.Stream()
    offset = rank * w.n_chains                             # weak scaling: disjoint chain-id ranges
    enqueue, sync_call, d2h_bytes = make_calls(R, torch, w, offset, stream)
    summary_dev = torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, n):
        """n calls of fn on `stream`, each bracketed by its own event pair; L2 flushed between calls
        outside the pairs. Returns per-call milliseconds."""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        with torch.cuda.stream(stream):
            for a, b in ev:
                flush.fill_(1)
                a.record(stream); fn(); b.record(stream)
        stream.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    # ---- device-timed leg ---------------------------------------------------------------------
    timed(lambda: enqueue(summary_dev), warmup)
    launches_per_step = R.rosen_last_launch_count()
    kernel_name = R.rosen_last_kernel_name()
    sampler = ClockSampler(local_rank); sampler.start()
    time.sleep(0.3)
    barrier()
    t0 = time.perf_counter()
    ms = timed(lambda: enqueue(summary_dev), steps)
    barrier()
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1)
    total_ms = sum(ms)
    extra = w.perm is not None or w.beta_eps is not None
    summary = sync_call() if extra else R.summary_from_device(summary_dev)

    # ---- dominant kernel alone (generation kernel, no second pass), live, same stream ------------
    timed(lambda: enqueue(None), 2)
    kms = timed(lambda: enqueue(None), max(3, min(steps, 10)))
    kernel_ms = sum(kms) / len(kms)

    dump_probe_conf = dump_probe_lnw = None
    if w.dump and w.kind == "realspace":
        dump_probe_conf = torch.empty((w.n_chains, w.N, 3), dtype=torch.float32, device="cuda")
        dump_probe_lnw = torch.empty((w.n_chains,), dtype=torch.float64, device="cuda")
    # ---- dump path (config 5): store phase D1 in situ = time(generation + dump) - time(generation only), same
    # launch geometry and lane mapping; bytes stored / that difference = achieved HBM write GB/s of the store phase
    dump_info = None
    if w.dump and w.kind == "realspace":
        def gen_only():
            R.rosen_realspace_generate_async(w.N, w.n_chains, w.k_trials, w.bond_len, w.sigma, w.seed, offset,
                                             outputs=None, summary_device=None, stream=stream)
        timed(gen_only, 1)
        t_gen = min(timed(gen_only, 3))
        t_all = min(kms)
        nbytes = w.n_chains * (12 * w.N + 8)
        diff = t_all - t_gen
        resolved = diff > 0.01 * t_all          # below 1 % of the call the difference is timing noise
        # the store phase alone: the same store routine, block size and grid over a resident synthetic chain (rosen_realspace_dump_probe)
        def probe():
            R.rosen_realspace_dump_probe(w.N, w.n_chains, dump_probe_conf, dump_probe_lnw, stream=stream)
        timed(probe, 2)
        t_probe = min(timed(probe, 5))
        dump_info = {"bytes_per_step": nbytes, "with_dump_ms": t_all, "generation_only_ms": t_gen, "store_phase_ms": diff,
                     "isolated_store_ms": t_probe, "isolated_store_GBps": nbytes / (t_probe * 1e-3) / 1e9,
                     "achieved_GBps": nbytes / (diff * 1e-3) / 1e9 if resolved else None,
                     "whole_call_GBps": nbytes / (t_all * 1e-3) / 1e9,
                     "note": None if resolved else "store phase not resolvable: hidden under generation (compute-bound call)"}

    # ---- end-to-end leg: synchronous C-ABI call, host buffers ------------------------------------
    for _ in range(2):
        sync_call()
    barrier()
    e0 = time.perf_counter()
    for _ in range(steps):
        s_host = sync_call()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - e0
    barrier()

    # ---- max over ranks ---------------------------------------------------------------------------
    if dist is not None:
        t = torch.tensor([total_ms, e2e_s, kernel_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, e2e_s, kernel_ms = (float(x) for x in t.cpu())
        parts = [None] * world
        dist.all_gather_object(parts, summary)
        summary = R.rosen_summary_merge(parts)             # rank order: deterministic
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    chains_total = w.n_chains * world
    value = chains_total * steps / (total_ms * 1e-3)
    steps_attempted = summary["n_steps_attempted"]
    peaks, peaks_src = load_measured_peaks()
    n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    sm_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    peak_winst = n_sm * 4 * sm_hz                           # 4 schedulers/SM, 1 warp-instruction/clk each
    alg_winst = algorithmic_thread_instr(w) * w.n_chains / 32.0
    achieved = alg_winst / (kernel_ms * 1e-3)
    if w.kind == "lattice" and w.N >= 193 and not extra:
        # hash-map kernel (DESIGN.md 5.5 / 6): ncu shows it issue-bound (67 % issue-active, 11 % of DRAM peak), so the
        # roofline is the issue peak; algorithmic work per ATTEMPTED step (not per nominal step: most long chains die
        # early): 3 cube look-ups (hash 8 + compare 6 each), 6 occupancy bits (4 each), count/choose 15, insert 10,
        # observables 12, weight 3, a quarter Philox block 17.5 = 123.5 thread-instructions
        alg_winst = HASH_INSTR_PER_STEP * (steps_attempted / world) / 32.0
        achieved = alg_winst / (kernel_ms * 1e-3)
    long_real = w.kind == "realspace" and w.N >= 400
    if long_real:
        # cell-list kernel (DESIGN.md 5.6 / 6), per ATTEMPTED step: k trials x (35 Philox + 45 direction + 7 x 3.2 candidate
        # pair tests) + 27 cell look-ups x 14 + ~40 listed monomers x 10 (candidate test) + 50 for count/choose/place/sums
        real_long_instr = w.k_trials * (80.0 + 7.0 * 3.2) + 27 * 14.0 + 40 * 10.0 + 50.0
        alg_winst = real_long_instr * (steps_attempted / world) / 32.0
        achieved = alg_winst / (kernel_ms * 1e-3)
    prof = profile_metrics(w)
    if extra:
        achieved = float("nan")
    roofline = {"bound": "alu", "achieved": achieved / 1e9, "peak": peak_winst / 1e9, "unit": "Gwarp-inst/s",
                "frac": achieved / peak_winst, "traffic": prof.get("traffic"), "kernel": kernel_name, "kernel_ms": kernel_ms,
                "peak_source": f"{n_sm} SMs x 4 schedulers x sm_max_mhz ({peaks_src} MEASURED_PEAKS.json)",
                "algorithmic_thread_instr_per_chain": algorithmic_thread_instr(w)}
    if w.kind == "lattice" and w.N >= 193 and not extra:
        del roofline["algorithmic_thread_instr_per_chain"]
        roofline["algorithmic_thread_instr_per_attempted_step"] = HASH_INSTR_PER_STEP
        roofline["note"] = "kernel_ms covers table memset + generation kernel + record reduction"
    if long_real:
        del roofline["algorithmic_thread_instr_per_chain"]
        roofline["algorithmic_thread_instr_per_attempted_step"] = real_long_instr
        roofline["note"] = "kernel_ms covers workspace memset + generation kernel + record reduction"
    if clocks.get("sm_mhz"):
        roofline["frac_at_measured_clock"] = achieved / (n_sm * 4 * clocks["sm_mhz"] * 1e6)
    if extra:
        alg_x, model_x = alg_warp_inst(w, steps_attempted / world)
        ach_x = alg_x / (kernel_ms * 1e-3)
        roofline = {"bound": "alu", "achieved": ach_x / 1e9, "peak": peak_winst / 1e9, "unit": "Gwarp-inst/s", "frac": ach_x / peak_winst,
                    "traffic": prof.get("traffic"), "kernel": kernel_name, "kernel_ms": kernel_ms, "model": model_x,
                    "peak_source": f"{n_sm} SMs x 4 schedulers x sm_max_mhz ({peaks_src} MEASURED_PEAKS.json)",
                    "note": "model / PERM workload (SURVEY.md 8(f) rows 4, 2): kernel_ms covers the generation kernel + record reduction"}
    if w.kind == "lattice" and w.N < 193 and not extra:
        # SURVEY.md 8(d) wrote "930 x ~5" per site test where DESIGN.md 6 counts the 6 equality tests of the method: both
        survey = 5.0 * lattice_site_tests(w.N) + 70.0 * ((w.N + 3) // 4) + 20.0 * (w.N - 1)
        roofline["frac_survey_coefficient"] = survey * w.n_chains / 32.0 / (kernel_ms * 1e-3) / peak_winst
        roofline["algorithmic_thread_instr_per_chain_survey"] = survey
    if prof.get("warp_inst_executed"):
        # "utilisation is not usefulness": what the kernel ISSUES per attempted step next to what the method needs
        roofline["issued_thread_instr_per_attempted_step"] = prof["warp_inst_executed"] * 32.0 / (steps_attempted / world)
        roofline["active_lane_ratio"] = prof.get("active_lane_ratio")
        roofline["issue_active_pct_ncu"] = prof.get("issue_active_pct")
        roofline["profile"] = prof.get("file")

    out = {
        "metric": METRIC, "value": value, "unit": "chains/s", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": total_ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32+f64" if w.kind == "lattice" else "f32+f64", "data": "synthetic",
        "config": {"workload": w.name, "kind": w.kind, "N": w.N, "n_chains_per_gpu": w.n_chains, "seed": w.seed,
                   "k_trials": w.k_trials, "bond_len": w.bond_len, "sigma": w.sigma, "dump": w.dump,
                   "parallelism": f"chain-range sharding x{world}, no collective",
                   "l2": "256 MiB buffer written between timed steps; the path reads no HBM input"},
        "monomer_steps_per_s": steps_attempted * steps / (total_ms * 1e-3),
        "monomer_steps_nominal_per_s": chains_total * (w.N - 1) * steps / (total_ms * 1e-3),
        "summary": {k: summary[k] for k in ("mean_ree2", "mean_rg2", "attrition", "ln_mean_W", "n_dead")},
        "clocks": clocks, "roofline": roofline,
        "e2e": {"value": chains_total * steps / e2e_s, "unit": "chains/s", "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": d2h_bytes, "ms_per_step": e2e_s / steps * 1e3,
                "note": "no input arrays exist (parameters by value); result = host rosen_summary"
                        + (" + host conf/lnW" if w.dump else "")},
        "gpu_launches": launches_per_step * steps,
    }
    if dump_info is not None:
        dump_info["peak_GBps"] = float(peaks.get("hbm_gbs", 6650.0))
        dump_info["frac"] = dump_info["achieved_GBps"] / dump_info["peak_GBps"] if dump_info["achieved_GBps"] else None
        dump_info["isolated_store_frac"] = dump_info["isolated_store_GBps"] / dump_info["peak_GBps"]
        out["dump_path"] = dump_info
    if world == 1 and not args.no_cpu_baseline:
        m, dt, _ = time_oracle(w, args.cpu_seconds / 2)
        cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
        per = max(16 if w.N <= 2048 else 1, int(m / dt * args.cpu_seconds / 2))   # ~cpu_seconds/2 of work per thread
        ma, dta = time_oracle_all_cores(w, per, cores)
        if w.kind == "realspace" and not extra:
            # decision parity on the single-thread sample: chains whose digest differs from the oracle's = flip fraction
            import numpy as np
            import oracle
            ref = oracle.realspace_generate(w.N, m, w.k_trials, w.bond_len, w.sigma, w.seed, chain_offset=offset, outputs=("digest",))
            _, tg = R.rosen_realspace_generate(w.N, m, w.k_trials, w.bond_len, w.sigma, w.seed, chain_offset=offset, outputs=("digest",))
            out["flip_fraction"] = {"value": float((tg["digest"].cpu().numpy().view(np.uint64) != ref.digest).mean()),
                                    "chains": m, "bar": 1e-4}
        out["cpu_baseline"] = {"value": ma / dta, "unit": "chains/s", "cores": cores, "kind": "oracle",
                               "sample": f"{cores} threads x {per} chains (disjoint chain-id ranges of {w.name}), {dta:.1f} s",
                               "single_thread": {"value": m / dt, "cores": 1,
                                                 "sample": f"chain ids [0, {m}) of {w.name}, {dt:.1f} s"}}
    if world == 1 and w.name == DEFAULT_WORKLOAD and not args.no_configs:
        # every other BASELINE configuration in the same process, after the headline leg, so
        # that the one line the driver records carries a number for each: configs 1, 3, 5 and the six points of config 4
        sampler2 = ClockSampler(local_rank); sampler2.start()
        c0 = time.perf_counter()
        block = {}
        for cw in (workloads.CONFIG_1, workloads.CONFIG_3, workloads.CONFIG_5, *workloads.CONFIG_4):
            block[cw.name] = measure_brief(R, torch, cw, stream, timed, peak_winst, float(peaks.get("hbm_gbs", 6650.0)),
                                           steps=max(5, min(steps, 10)), flip_sample=0 if args.no_cpu_baseline else 1 << 13)
            torch.cuda.empty_cache()
        c1 = time.perf_counter()
        out["configs"] = block
        out["configs_clocks"] = sampler2.stop(c0, c1)
        out["configs_wall_s"] = c1 - c0
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE config 4: lattice length sweep N in {8..256}, 2^24 chains each, seed 11: attrition(N), nu from
    <Ree2> ~ (N-1)^(2 nu) (least squares on logs, reading A14), throughput per N. One JSON line."""
    import math

    import torch
    import paper_1704_04381_b200 as R
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    R.load_library()
    stream = torch.cuda.Stream()
    summary_dev = torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda")
    rows = []
    for w in workloads.CONFIG_4:
        def call():
            R.rosen_lattice_generate_async(w.N, w.n_chains, w.seed, 0, outputs=None, summary_device=summary_dev, stream=stream)
        ms = []
        with torch.cuda.stream(stream):
            for i in range(2 + max(args.steps, 1)):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream); call(); b.record(stream)
                ms.append((a, b))
        stream.synchronize()
        t = [a.elapsed_time(b) for a, b in ms][2:]
        sm = R.summary_from_device(summary_dev)
        best = min(t)
        rows.append({"N": w.N, "ms": best, "chains_per_s": w.n_chains / (best * 1e-3),
                     "monomer_steps_per_s": sm["n_steps_attempted"] / (best * 1e-3), "attrition": sm["attrition"],
                     "mean_ree2": sm["mean_ree2"], "mean_rg2": sm["mean_rg2"], "ln_mean_W": sm["ln_mean_W"],
                     "ess_fraction": sm["sum_w"] ** 2 / sm["sum_w2"] / sm["n_chains"], "kernel": R.rosen_last_kernel_name()})
    fit = R.rosen_fit_exponents([r["N"] for r in rows], [r["mean_ree2"] for r in rows], [r["ln_mean_W"] for r in rows],
                                use_steps=True)                    # Eq. 4-7, x = N - 1 (reading A14)
    slope, mu = 2.0 * fit["nu"], fit["mu"]
    print(json.dumps({"metric": "lattice length sweep (BASELINE config 4)", "seed": workloads.CONFIG_4[0].seed,
                      "n_chains": workloads.CONFIG_4[0].n_chains, "nu_fit": slope / 2.0, "mu_fit": mu, "gamma_fit": fit["gamma"], "fit": fit,
                      "sweep": rows, "data": "synthetic"}))


# The paper's own benchmark (Tables 1-2): wall time to generate 10^6 chains of N monomers, for the lengths its
# tables list. Its chains are restarted on dead ends, so its times are per 10^6 FULL-LENGTH chains; here dead chains are kept
# (reading A6), so both the time per 10^6 attempts and that time divided by the surviving fraction are reported.
PAPER_TABLE_N = (4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048, 100, 500, 1000, 2500, 5000, 10000)
PAPER_TABLE1_GTX1080_S = {4: 0.00324, 8: 0.00901, 16: 0.02664, 32: 0.09192, 64: 0.38830, 128: 1.73263, 256: 7.50125, 512: 49.8232,
                          1024: 373.824, 2048: 3981.55, 100: 8.1, 500: 14.5, 1000: 559.9, 2500: 3574.0, 5000: 14088.0, 10000: 55883.1}
PAPER_TABLE2_GTX1080_S = {4: 0.16288, 8: 0.44877, 16: 2.31603, 32: 11.4375, 64: 58.3319, 128: 226.441, 256: 986.501, 512: 5905.82,
                          1024: 45513.8, 2048: 378758.0}


def run_paper_tables(args):
    """`--paper-tables`: 10^6 chains per length of Tables 1-2 (lattice; real space with k = 16, b = sigma = 1 -- the paper
    does not state its trial set -- and with k = 64, sigma = 0.8 for the long lengths where the former lets no chain
    survive). One JSON line; times are device-timed, best of 3, summary-only calls."""
    import torch
    import paper_1704_04381_b200 as R
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    R.load_library()
    stream = torch.cuda.Stream()
    summary_dev = torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda")
    n = 1000000

    def timed(call):
        ev = []
        with torch.cuda.stream(stream):
            for _ in range(4):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream); call(); b.record(stream)
                ev.append((a, b))
        stream.synchronize()
        return min(a.elapsed_time(b) for a, b in ev[1:]) * 1e-3

    def row(N, sec, paper):
        sm = R.summary_from_device(summary_dev)
        alive = 1.0 - sm["attrition"]
        return {"N": N, "s_per_1e6_attempts": sec, "alive_fraction": alive,
                "s_per_1e6_full_length": sec / alive if alive > 0 else None, "paper_gtx1080_s": paper,
                "monomer_steps_per_s": sm["n_steps_attempted"] / sec, "kernel": R.rosen_last_kernel_name()}

    lattice, real16, real64 = [], [], []
    for N in PAPER_TABLE_N:
        sec = timed(lambda: R.rosen_lattice_generate_async(N, n, 1, 0, outputs=None, summary_device=summary_dev, stream=stream))
        lattice.append(row(N, sec, PAPER_TABLE1_GTX1080_S.get(N)))
    for N in PAPER_TABLE_N:
        sec = timed(lambda: R.rosen_realspace_generate_async(N, n, 16, 1.0, 1.0, 1, 0, outputs=None, summary_device=summary_dev, stream=stream))
        real16.append(row(N, sec, PAPER_TABLE2_GTX1080_S.get(N)))
    for N in (512, 1024, 2048, 2500, 5000, 10000):
        m = n // 10                                                    # 10^5 chains, scaled to 10^6
        sec = timed(lambda: R.rosen_realspace_generate_async(N, m, 64, 1.0, 0.8, 1, 0, outputs=None, summary_device=summary_dev, stream=stream))
        r = row(N, sec * 10.0, PAPER_TABLE2_GTX1080_S.get(N))
        r["note"] = "10^5 chains timed, x10"
        real64.append(r)
    print(json.dumps({"metric": "seconds per 10^6 chains at the lengths of the paper's Tables 1-2 (PAPER.md:266-320)", "n_chains": n,
                      "lattice": lattice, "realspace_k16_sigma1": real16, "realspace_k64_sigma0.8": real64, "data": "synthetic"}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(workloads.CONFIGS))
    ap.add_argument("--impl", default="product", choices=("product", "reference"))
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="default workload only: skip the block that times every other BASELINE config")
    ap.add_argument("--sweep", action="store_true", help="run BASELINE config 4 (length sweep) instead")
    ap.add_argument("--paper-tables", action="store_true", help="10^6 chains at every length of the paper's Tables 1-2 instead")
    args = ap.parse_args()
    w = workloads.CONFIGS[args.workload]
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started without torchrun: launch the N ranks ourselves (one process per GPU), never measure 1 GPU as N
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                  f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1", "--master-port", str(port),
                                  os.path.abspath(__file__)] + sys.argv[1:])
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch with torchrun --nproc-per-node {args.gpus}")
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.sweep:
        if rank == 0:
            run_sweep(args)
        return
    if args.paper_tables:
        if rank == 0:
            run_paper_tables(args)
        return
    if args.impl == "reference":
        run_reference(args, w, rank)
    else:
        run_product(args, w, rank, world, local_rank)


if __name__ == "__main__":
    main()

"""GPU parity: CUDA lattice path (through the C ABI) vs the CPU oracle, element by element.

Bar (BASELINE north_star): trajectory, m_i sequence, dead/alive flag bit-exact per chain; ensemble
fp64 sums within 1e-12 relative.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1704_04381_b200 import workloads

pytestmark = pytest.mark.gpu

REL = 1e-12
ALL = ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")


@pytest.fixture(scope="module")
def R():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1704_04381_b200 as R
    R.load_library()
    return R


def compare_per_chain(t, o, N):
    conf = t["conf"].cpu().numpy()
    assert np.array_equal(conf, o.conf), "trajectory mismatch"
    assert np.array_equal(t["m_seq"].cpu().numpy(), o.m_seq), "m sequence mismatch"
    assert np.array_equal(t["alive"].cpu().numpy(), o.alive), "alive flag mismatch"
    assert np.array_equal(t["digest"].cpu().numpy().view(np.uint64), o.digest), "digest mismatch"
    lnW = t["lnW"].cpu().numpy()
    dead = o.alive == 0
    assert np.all(np.isneginf(lnW[dead]))
    assert np.allclose(lnW[~dead], o.lnW[~dead], rtol=REL, atol=0)
    assert np.array_equal(t["ree2"].cpu().numpy(), o.ree2)          # integers: exact
    assert np.allclose(t["rg2"].cpu().numpy(), o.rg2, rtol=REL, atol=0)


def compare_summary(s, so):
    for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
        assert s[key] == so[key], key
    for key in ("ln_shift", "sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "attrition", "ln_mean_W"):
        assert math.isclose(s[key], so[key], rel_tol=REL, abs_tol=0.0), (key, s[key], so[key])


def test_config1_full_parity(R):
    w = workloads.CONFIG_1
    s, t = R.rosen_lattice_generate(w.N, w.n_chains, w.seed, outputs=ALL)
    o = oracle.lattice_generate(w.N, w.n_chains, w.seed)
    compare_per_chain(t, o, w.N)
    compare_summary(s, o.summary)
    assert "lattice" in R.rosen_last_kernel_name() and R.rosen_last_launch_count() == 2


@pytest.mark.parametrize("N,n_chains,seed,offset", [
    (2, 1, 0, 0), (2, 1000, 5, 7), (3, 33, 1, 0), (4, 257, 2, 0), (5, 4099, 3, 1 << 40),
    (9, 5000, 4, (1 << 32) - 100), (17, 3001, 8, 0), (33, 2049, 9, 0), (64, 9001, 7, 12345),
    (65, 777, 7, 0), (127, 1500, 11, 0), (128, 1500, 11, 0), (129, 700, 11, 0), (200, 900, 12, 0),
    (256, 1200, 11, 3), (300, 300, 13, 0), (512, 200, 14, 0),
])
def test_shapes_ragged_and_edges(R, N, n_chains, seed, offset):
    s, t = R.rosen_lattice_generate(N, n_chains, seed, chain_offset=offset, outputs=ALL)
    o = oracle.lattice_generate(N, n_chains, seed, chain_offset=offset)
    compare_per_chain(t, o, N)
    compare_summary(s, o.summary)


# Long chains (N > ROSEN_LATTICE_SCAN_MAX_N = 512): the hash-set kernel of lattice_hash.cu, the range of the paper's
# "global-memory version" (Table 1). Same bit-exact bar as the scan kernel. Sizes keep the oracle's
# O(N^2) scan to seconds; N = 1366 is the first length of the 4096-slot table, 1365 the fullest 2048-slot one.
@pytest.mark.parametrize("N,n_chains,seed,offset", [
    (513, 1000, 14, 0), (1024, 777, 15, 5), (1365, 300, 16, 0), (1366, 300, 16, 0), (2048, 400, 17, 1 << 33),
    (4096, 257, 18, 0), (10000, 200, 19, 0), (16383, 100, 20, 0),
])
def test_long_chains_hash_kernel(R, N, n_chains, seed, offset):
    s, t = R.rosen_lattice_generate(N, n_chains, seed, chain_offset=offset, outputs=ALL)
    assert "lattice_hash_kernel" in R.rosen_last_kernel_name() and R.rosen_last_launch_count() == 5
    o = oracle.lattice_generate(N, n_chains, seed, chain_offset=offset)
    compare_per_chain(t, o, N)
    compare_summary(s, o.summary)
    s2, _ = R.rosen_lattice_generate(N, n_chains, seed, chain_offset=offset)          # summary-only variant
    for k in s:
        if not k.startswith("digest"):
            assert s[k] == s2[k], k


def test_scan_kernel_over_its_whole_range(R, monkeypatch):
    """By default N >= ROSEN_LATTICE_HASH_MIN_N = 193 takes the hash-map kernel; the knob lattice_hash_min_n = 513 keeps the
    scan kernel up to its limit N = 512 so that its wide variant stays covered against the oracle."""
    R.rosen_debug_set("lattice_hash_min_n", 513)
    for N, n, seed in [(193, 800, 12), (256, 1200, 11), (300, 300, 13), (512, 200, 14)]:
        s, t = R.rosen_lattice_generate(N, n, seed, outputs=ALL)
        assert "lattice_dp_kernel<wide" in R.rosen_last_kernel_name()
        o = oracle.lattice_generate(N, n, seed)
        compare_per_chain(t, o, N)
        compare_summary(s, o.summary)
    R.rosen_debug_set("lattice_hash_min_n", 0)
    R.rosen_lattice_generate(192, 100, 1)
    assert "lattice_dp_kernel" in R.rosen_last_kernel_name()
    R.rosen_lattice_generate(193, 100, 1)
    assert "lattice_hash_kernel" in R.rosen_last_kernel_name() and R.rosen_last_launch_count() == 3


def test_hash_kernel_equals_scan_kernel_on_short_chains(R, monkeypatch):
    """The knob lattice_hash_min_n = 2 routes short chains through the hash kernel: it must reproduce the scan kernel
    (and with it the oracle and its enumeration pins) bit for bit, per chain and in the ensemble sums, with
    many chains per lane (table generations) and more chains than resident threads."""
    import torch
    for N, n, seed in [(16, 1 << 16, 1), (64, 400000, 7), (200, 30011, 3)]:
        R.rosen_debug_set("lattice_hash_min_n", 513)
        s_scan, t_scan = R.rosen_lattice_generate(N, n, seed, outputs=ALL)
        assert "lattice_dp_kernel" in R.rosen_last_kernel_name()
        R.rosen_debug_set("lattice_hash_min_n", 2)
        s_hash, t_hash = R.rosen_lattice_generate(N, n, seed, outputs=ALL)
        assert "lattice_hash_kernel" in R.rosen_last_kernel_name()
        for k in ALL:
            if k == "lnW":      # N <= 64: the scan kernel sums an m histogram, the hash kernel adds step by step
                assert torch.equal(torch.isinf(t_scan[k]), torch.isinf(t_hash[k]))
                assert torch.allclose(t_scan[k], t_hash[k], rtol=REL, atol=0.0), (N, k)
            else:
                assert torch.equal(t_scan[k], t_hash[k]), (N, k)
        for k in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
            assert s_scan[k] == s_hash[k], k
        for k in ("sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "ln_mean_W"):
            assert math.isclose(s_scan[k], s_hash[k], rel_tol=REL), k
    R.rosen_debug_set("lattice_hash_min_n", 0)
    assert R.rosen_workspace_bytes() > (1 << 20)
    assert R.rosen_workspace_release() == R.ROSEN_OK


def test_long_chain_properties_at_bench_size(R):
    """N = 1024, 2^18 chains in the launch configuration bench.py --workload lattice_long times: invariants that
    hold at any size plus sampled chains recomputed one by one by the oracle (chain_offset sub-ranges)."""
    import torch
    N, n, seed = 1024, 1 << 18, 23
    s, t = R.rosen_lattice_generate(N, n, seed, outputs=("lnW", "alive", "ree2", "rg2", "digest"))
    alive = t["alive"].bool()
    assert s["n_dead"] == int((~alive).sum()) and 0.1 < s["attrition"] < 0.35
    assert bool(torch.isinf(t["lnW"][~alive]).all()) and bool((t["ree2"][~alive] == 0).all())
    L = s["ln_shift"]
    assert bool((t["lnW"][alive] <= math.log(6.0) + (N - 2) * math.log(5.0) + 1e-9).all()) and L == float(t["lnW"][alive].max()) and bool((t["ree2"][alive] <= (N - 1) ** 2).all())
    assert bool((t["ree2"][alive] % 2 == (N - 1) % 2).all())           # bipartite lattice: parity of |r|^2 = parity of the step count
    for off in (0, 77777, n - 3):
        o = oracle.lattice_generate(N, 3, seed, chain_offset=off)
        assert np.array_equal(t["digest"][off:off + 3].cpu().numpy().view(np.uint64), o.digest)
        assert np.array_equal(t["ree2"][off:off + 3].cpu().numpy(), o.ree2)
        assert np.allclose(t["lnW"][off:off + 3].cpu().numpy(), o.lnW, rtol=REL, atol=0)
    s2, _ = R.rosen_lattice_generate(N, n, seed)
    for k in s:
        if not k.startswith("digest"):
            assert s[k] == s2[k], k


def test_summary_only_variant_is_bit_identical_and_deterministic(R):
    N, n, seed = 64, 100003, 7
    s0, _ = R.rosen_lattice_generate(N, n, seed)
    s1, _ = R.rosen_lattice_generate(N, n, seed)
    assert s0 == s1
    s2, t = R.rosen_lattice_generate(N, n, seed, outputs=("lnW", "ree2", "rg2", "alive"))
    for k in s0:
        if not k.startswith("digest"):
            assert s0[k] == s2[k], k
    s3, _ = R.rosen_lattice_generate(N, n, seed, outputs=ALL)
    for k in s0:
        if not k.startswith("digest"):
            assert s0[k] == s3[k], k
    o = oracle.lattice_generate(N, n, seed, outputs=("digest",))
    compare_summary(s3, o.summary)


def test_host_outputs_and_dump_entry_points(R):
    N, n, seed = 24, 5000, 21
    s_d, t_d = R.rosen_lattice_generate(N, n, seed, outputs=ALL)
    s_h, t_h = R.rosen_lattice_generate(N, n, seed, outputs=ALL, host_outputs=True)
    assert s_d == s_h
    for k in ALL:
        assert not t_h[k].is_cuda
        assert np.array_equal(t_d[k].cpu().numpy(), t_h[k].numpy()), k
    s, conf, lnW = R.rosen_lattice_dump(N, n, seed)
    assert np.array_equal(conf.cpu().numpy(), t_d["conf"].cpu().numpy())
    assert np.array_equal(lnW.cpu().numpy(), t_d["lnW"].cpu().numpy())


def test_chain_offset_subrange_and_merge(R):
    N, n, seed = 32, 40000, 5
    s_all, t_all = R.rosen_lattice_generate(N, n, seed, outputs=("digest", "lnW"))
    parts = []
    for rank in range(3):
        off, cnt = workloads.shard(n, rank, 3)
        s, t = R.rosen_lattice_generate(N, cnt, seed, chain_offset=off, outputs=("digest", "lnW"))
        assert np.array_equal(t["digest"].cpu().numpy(), t_all["digest"][off:off + cnt].cpu().numpy())
        parts.append(s)
    m = R.rosen_summary_merge(parts)
    for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
        assert m[key] == s_all[key]
    for key in ("sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "ln_mean_W"):
        assert math.isclose(m[key], s_all[key], rel_tol=1e-13)


def test_error_codes(R):
    for args, code in [((1, 10, 0), R.ROSEN_EINVAL), ((8, 0, 0), R.ROSEN_EINVAL), ((16384, 10, 0), R.ROSEN_ERANGE)]:
        with pytest.raises(R.RosenError) as e:
            R.rosen_lattice_generate(*args)
        assert e.value.code == code


def test_config2_full_size_sampled(R):
    """BASELINE config 2 at full size in the launch configuration bench.py times (summary only),
    plus the same launch with per-chain scalars for sampled one-by-one oracle checks and
    size-independent properties."""
    import torch
    w = workloads.CONFIG_2
    s_bench, _ = R.rosen_lattice_generate(w.N, w.n_chains, w.seed)
    name_bench = R.rosen_last_kernel_name()
    s, t = R.rosen_lattice_generate(w.N, w.n_chains, w.seed, outputs=("lnW", "alive", "ree2", "rg2", "digest"))
    for k in s_bench:
        if not k.startswith("digest"):
            assert s_bench[k] == s[k], k                      # same reduction tree, bit-identical
    assert name_bench.startswith("lattice")
    # contiguous prefix + scattered samples, one by one against the oracle
    pre = 1 << 15
    o = oracle.lattice_generate(w.N, pre, w.seed, outputs=("lnW", "alive", "ree2", "rg2", "digest"))
    assert np.array_equal(t["digest"][:pre].cpu().numpy().view(np.uint64), o.digest)
    assert np.array_equal(t["alive"][:pre].cpu().numpy(), o.alive)
    assert np.array_equal(t["ree2"][:pre].cpu().numpy(), o.ree2)
    rng = np.random.default_rng(2024)
    ids = np.unique(np.concatenate([rng.integers(0, w.n_chains, 2000), [w.n_chains - 1, w.n_chains - 2]]))
    dg = t["digest"].cpu().numpy().view(np.uint64); lw = t["lnW"].cpu().numpy(); rg = t["rg2"].cpu().numpy()
    for i in ids:
        oi = oracle.lattice_generate(w.N, 1, w.seed, chain_offset=int(i), outputs=("lnW", "rg2", "digest"))
        assert oi.digest[0] == dg[i]
        assert (np.isneginf(lw[i]) and np.isneginf(oi.lnW[0])) or math.isclose(lw[i], oi.lnW[0], rel_tol=REL)
        assert math.isclose(rg[i], oi.rg2[0], rel_tol=REL)
    # properties at full size: the summary is the reduction of the per-chain outputs
    alive = t["alive"].bool()
    wgt = torch.where(alive, torch.exp(t["lnW"] - s["ln_shift"]), torch.zeros_like(t["lnW"]))
    assert int((~alive).sum()) == s["n_dead"]
    assert math.isclose(float(wgt.sum()), s["sum_w"], rel_tol=1e-11)
    assert math.isclose(float((wgt * t["ree2"]).sum()), s["sum_w_ree2"], rel_tol=1e-11)
    assert math.isclose(float((wgt * t["rg2"]).sum()), s["sum_w_rg2"], rel_tol=1e-11)
    d64 = t["digest"]
    assert int(d64.sum()) & (2 ** 64 - 1) == s["digest_sum"]     # int64 wrap-around sum == uint64 sum mod 2^64
    # physics sanity (loose): attrition ~3.6e-3, nu-consistent <Ree2> ~ 152
    assert 2e-3 < s["attrition"] < 6e-3 and 140 < s["mean_ree2"] < 165


def test_config4_sweep_reduced(R):
    """BASELINE config 4 (length sweep, seed 11) at 2^18 chains per N: kernel variant per N, sampled per-chain
    parity against the oracle, attrition grows with N, nu from <Ree2> ~ (N-1)^(2 nu) in the paper's band
    (PAPER.md:350 0.601 text / :374 0.588 table; [0.58, 0.62])."""
    n = 1 << 18
    xs, ys, att = [], [], []
    for N in workloads.CONFIG_4_N:
        s, t = R.rosen_lattice_generate(N, n, 11, outputs=("digest", "lnW", "alive", "ree2"))
        name = R.rosen_last_kernel_name()
        if N >= 193:
            assert name.startswith("lattice_hash_kernel")
        else:
            assert name.startswith("lattice_dp_kernel<wide") if N > 128 else name.startswith("lattice_dp_kernel") and "wide" not in name
        pre = 384
        o = oracle.lattice_generate(N, pre, 11, outputs=("digest", "lnW", "alive", "ree2"))
        assert np.array_equal(t["digest"][:pre].cpu().numpy().view(np.uint64), o.digest)
        assert np.array_equal(t["alive"][:pre].cpu().numpy(), o.alive)
        assert np.array_equal(t["ree2"][:pre].cpu().numpy(), o.ree2)
        tail = oracle.lattice_generate(N, 2, 11, chain_offset=n - 2, outputs=("digest",))
        assert np.array_equal(t["digest"][n - 2:].cpu().numpy().view(np.uint64), tail.digest)
        xs.append(math.log(N - 1)); ys.append(math.log(s["mean_ree2"])); att.append(s["attrition"])
    assert att[0] == 0.0 and all(a <= b for a, b in zip(att, att[1:])) and 0.02 < att[-1] < 0.06
    mx, my = sum(xs) / len(xs), sum(ys) / len(ys)
    nu = 0.5 * sum((x - mx) * (y - my) for x, y in zip(xs, ys)) / sum((x - mx) ** 2 for x in xs)
    assert 0.57 < nu < 0.63, nu


def test_long_chain_workspace_reuse_without_clearing(R):
    """The long-chain tables are cleared only on allocation or layout change (generation counters persist across calls):
    repeated calls of one layout, with other layouts and the real-space long kernel in between, reproduce the same chains."""
    ref = None
    for rep in range(4):
        s, t = R.rosen_lattice_generate(700, 3000, 23, outputs=("digest", "lnW"))
        assert R.rosen_last_kernel_name().startswith("lattice_hash_kernel")
        cur = (t["digest"].cpu().numpy().copy(), s["sum_w"], s["n_dead"])
        if ref is None:
            o = oracle.lattice_generate(700, 300, 23, outputs=("digest",))
            assert np.array_equal(cur[0][:300].view(np.uint64), o.digest)
            ref = cur
        assert np.array_equal(cur[0], ref[0]) and cur[1] == ref[1] and cur[2] == ref[2]
        if rep == 1:
            R.rosen_lattice_generate(1500, 500, 1)                     # another layout in between
        if rep == 2:
            s2, t2 = R.rosen_realspace_generate(450, 64, 16, 1.0, 0.8, 5, outputs=("digest",))
            o2 = oracle.realspace_generate(450, 64, 16, 1.0, 0.8, 5, outputs=("digest",))
            assert np.array_equal(t2["digest"].cpu().numpy().view(np.uint64), o2.digest)


def test_concurrent_calls_from_threads_and_streams(R):
    """Calls of one device share scratch (block partials, records, tables): the library serialises host threads and orders
    the streams itself, so concurrent callers get the results of sequential calls."""
    import threading
    import torch
    jobs = [(48, 30000, 100 + i) for i in range(4)] + [(300, 2000, 200 + i) for i in range(2)]
    want = [R.rosen_lattice_generate(N, n, seed, outputs=("digest",)) for N, n, seed in jobs]
    got = [None] * len(jobs)

    def run(i):
        N, n, seed = jobs[i]
        st = torch.cuda.Stream()
        for _ in range(3):
            got[i] = R.rosen_lattice_generate(N, n, seed, outputs=("digest",), stream=st)

    th = [threading.Thread(target=run, args=(i,)) for i in range(len(jobs))]
    for t in th: t.start()
    for t in th: t.join()
    for (s0, t0), (s1, t1) in zip(want, got):
        assert s0 == s1 and torch.equal(t0["digest"], t1["digest"])


def test_workspace_release_while_other_threads_call(R):
    """rosen_workspace_release takes the same per-device lock as the generate calls: a release issued while another host
    thread is inside a long-chain / model call waits for that call instead of freeing the tables its kernel is about to use."""
    import threading
    import torch
    jobs = [(300, 3000, 300), (1024, 500, 301)]
    want = [R.rosen_lattice_generate(N, n, seed, outputs=("digest", "lnW")) for N, n, seed in jobs]
    got = [[] for _ in jobs]
    stop = threading.Event()

    def run(i):
        N, n, seed = jobs[i]
        st = torch.cuda.Stream()
        for _ in range(12):
            got[i].append(R.rosen_lattice_generate(N, n, seed, outputs=("digest", "lnW"), stream=st))

    def release():
        while not stop.is_set():
            assert R.rosen_workspace_release() == R.ROSEN_OK

    th = [threading.Thread(target=run, args=(i,)) for i in range(len(jobs))]
    rel = threading.Thread(target=release)
    rel.start()
    for t in th: t.start()
    for t in th: t.join()
    stop.set(); rel.join()
    for (s0, t0), runs in zip(want, got):
        assert len(runs) == 12
        for s1, t1 in runs:
            assert s0 == s1 and torch.equal(t0["digest"], t1["digest"]) and torch.equal(t0["lnW"], t1["lnW"])
    assert R.rosen_workspace_release() == R.ROSEN_OK
    s2, t2 = R.rosen_lattice_generate(*jobs[1], outputs=("digest", "lnW"))       # everything released is made again
    assert s2 == want[1][0] and torch.equal(t2["digest"], want[1][1]["digest"])


def test_generation_counter_wrap_of_the_hash_kernel(R):
    """Every thread of the hash-map kernel tags its table entries with a generation counter that persists across calls; when
    it passes its largest value the thread clears its table and restarts at 1 (lattice_hash.cu). Reaching that naturally takes
    2^25 chains per thread: rosen_debug_set("generations_left", g) presets the counters so that it happens g chains from now,
    in the middle of a call whose tables are full of entries of the generations just below the limit."""
    import torch
    R.rosen_debug_set("hash_blocks_per_sm", 1)       # 148 x 256 resident threads: every thread grows ~5 chains of the call,
    N, n, seed = 600, 200000, 41                     # so the wrap falls between chains, on a table full of this call's entries
    s0, t0 = R.rosen_lattice_generate(N, n, seed, outputs=("digest", "lnW", "alive"))
    assert "lattice_hash_kernel" in R.rosen_last_kernel_name()
    o = oracle.lattice_generate(N, 3000, seed, outputs=("digest",))
    assert np.array_equal(t0["digest"][:3000].cpu().numpy().view(np.uint64), o.digest)
    for left in (0, 1, 2, 4):
        R.rosen_debug_set("generations_left", left)
        s1, t1 = R.rosen_lattice_generate(N, n, seed, outputs=("digest", "lnW", "alive"))
        assert s1 == s0, left
        for k in t0:
            assert torch.equal(t0[k], t1[k]), (left, k)
    s2, _ = R.rosen_lattice_generate(N, n, seed, outputs=("digest", "lnW", "alive"))      # and the calls after the wrap
    assert s2 == s0
    R.rosen_workspace_release()
    with pytest.raises(R.RosenError):
        R.rosen_debug_set("generations_left", 1)     # no workspace: refused, nothing to preset

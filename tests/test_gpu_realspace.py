"""GPU parity: CUDA real-space path (through the C ABI) vs the CPU oracle.

Bar (BASELINE north_star): coordinates within 1e-5 absolute in fp32 (expected: identical bits,
the arithmetic is specified to the operation), fraction of chains whose overlap decision flips
< 1e-4 (expected 0; measured via the per-chain decision digest), ensemble averages within 1e-6.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1704_04381_b200 import workloads

pytestmark = pytest.mark.gpu

ALL = ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")


@pytest.fixture(scope="module")
def R():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1704_04381_b200 as R
    R.load_library()
    return R


def check(R, N, n, k, b, sigma, seed, offset=0, exact=True):
    s, t = R.rosen_realspace_generate(N, n, k, b, sigma, seed, chain_offset=offset, outputs=ALL)
    o = oracle.realspace_generate(N, n, k, b, sigma, seed, chain_offset=offset)
    dg = t["digest"].cpu().numpy().view(np.uint64)
    flips = float((dg != o.digest).mean())
    assert flips < 1e-4, f"flip fraction {flips}"
    same = dg == o.digest
    conf = t["conf"].cpu().numpy()
    assert np.abs(conf[same] - o.conf[same]).max(initial=0.0) <= 1e-5
    if exact:   # by construction the two sides execute the same IEEE operations
        assert flips == 0.0
        assert np.array_equal(conf, o.conf)
        assert np.array_equal(t["m_seq"].cpu().numpy(), o.m_seq)
        assert np.array_equal(t["alive"].cpu().numpy(), o.alive)
        lnW = t["lnW"].cpu().numpy()
        dead = o.alive == 0
        assert np.all(np.isneginf(lnW[dead])) and np.allclose(lnW[~dead], o.lnW[~dead], rtol=1e-13, atol=0)
        assert np.allclose(t["ree2"].cpu().numpy(), o.ree2, rtol=1e-12, atol=0)
        assert np.allclose(t["rg2"].cpu().numpy(), o.rg2, rtol=1e-9, atol=0)
        for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
            assert s[key] == o.summary[key], key
    for key in ("sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "ln_mean_W"):
        both_nan = math.isnan(s[key]) and math.isnan(o.summary[key])      # every chain dead: 0/0 on both sides
        assert both_nan or math.isclose(s[key], o.summary[key], rel_tol=1e-6), (key, s[key], o.summary[key])
    return flips


def test_config3_prefix(R):
    w = workloads.CONFIG_3
    check(R, w.N, 1 << 13, w.k_trials, w.bond_len, w.sigma, w.seed)


def test_config5_prefix(R):
    w = workloads.CONFIG_5
    check(R, w.N, 192, w.k_trials, w.bond_len, w.sigma, w.seed)


@pytest.mark.parametrize("N,n,k,b,sigma,seed,offset", [
    (2, 1, 1, 1.0, 1.0, 0, 0), (2, 100, 5, 1.0, 1.0, 1, 0), (3, 3000, 16, 1.0, 1.0, 3, 0),
    (8, 1000, 1, 1.0, 0.5, 4, 0), (8, 1000, 2, 1.0, 0.9, 4, 9), (9, 777, 3, 1.5, 1.0, 5, 0),
    (16, 1001, 4, 1.0, 1.0, 6, 0), (16, 999, 7, 0.7, 1.0, 6, (1 << 32) - 5), (20, 600, 8, 1.0, 1.2, 7, 0),
    (33, 500, 9, 1.0, 1.0, 8, 0), (33, 500, 16, 1.0, 0.0, 8, 0), (40, 400, 17, 1.0, 1.0, 9, 0),
    (40, 300, 32, 2.0, 1.7, 9, 0), (31, 300, 33, 1.0, 1.0, 10, 0), (25, 300, 64, 1.0, 1.0, 10, 0),
    (25, 200, 65, 1.0, 0.8, 11, 0), (20, 150, 128, 1.0, 1.0, 11, 0), (18, 100, 129, 1.0, 1.0, 12, 0),
    (12, 100, 255, 1.0, 1.0, 12, 0), (130, 64, 16, 1.0, 1.0, 13, 0), (64, 2000, 16, 1.0, 1.9, 14, 0),
    (1024, 6, 4, 1.0, 0.6, 15, 0), (1024, 3, 2, 0.5, 0.0, 15, 2), (2048, 3, 3, 1.0, 0.5, 16, 1),   # ROSEN_REALSPACE_MAX_N
])
def test_shapes_ragged_and_edges(R, N, n, k, b, sigma, seed, offset):
    check(R, N, n, k, b, sigma, seed, offset)


def test_scan_kernel_over_its_whole_range(R, monkeypatch):
    """By default N >= ROSEN_REALSPACE_CELL_MIN_N = 400 takes the cell-list kernel; the knob realspace_cell_min_n = 2049 keeps
    the shared-memory scan kernel up to its limit so that its long-chain variants stay covered against the oracle."""
    R.rosen_debug_set("realspace_cell_min_n", 2049)
    for args in [(400, 20, 16, 1.0, 1.0, 13, 0), (1024, 6, 4, 1.0, 0.6, 15, 0), (1024, 3, 2, 0.5, 0.0, 15, 2), (2048, 3, 3, 1.0, 0.5, 16, 1)]:
        check(R, *args)
        assert R.rosen_last_kernel_name().startswith("realspace_kernel")
    R.rosen_debug_set("realspace_cell_min_n", 0)
    R.rosen_realspace_generate(399, 10, 4, 1.0, 0.5, 1)
    assert R.rosen_last_kernel_name().startswith("realspace_kernel")
    R.rosen_realspace_generate(400, 10, 4, 1.0, 0.5, 1)
    assert R.rosen_last_kernel_name().startswith("realspace_long_kernel") and R.rosen_last_launch_count() == 3


# Long chains (N > ROSEN_REALSPACE_SCAN_MAX_N = 2048): the cell-list kernel of realspace_long.cu, the range of the
# paper's real-space "global-memory version" (Table 2). Same bars as the shared-memory kernel.
@pytest.mark.parametrize("N,n,k,b,sigma,seed,offset", [
    (2049, 12, 8, 1.0, 0.6, 21, 0), (2500, 6, 32, 1.0, 1.0, 22, 3), (3000, 8, 2, 0.5, 0.0, 23, 0),
    (4096, 3, 65, 1.0, 0.8, 24, 1 << 34), (5000, 4, 16, 2.0, 1.0, 25, 0), (10000, 3, 4, 1.0, 0.0, 26, 0),
    (10000, 1, 24, 1.0, 0.4, 28, 0), (16383, 1, 16, 1.0, 0.3, 27, 0),        # chosen so that chains reach full length
])
def test_long_chains_cell_list_kernel(R, N, n, k, b, sigma, seed, offset):
    check(R, N, n, k, b, sigma, seed, offset)
    assert "realspace_long_kernel" in R.rosen_last_kernel_name() and R.rosen_last_launch_count() == 5


def test_cell_list_workspace_reuse_across_neighbouring_lengths(R):
    """N = 1000 (n_pad 1000) and N = 1001 (n_pad 1008) round to the same 32256-byte slice per warp but put the cell table at
    different offsets: the workspace must be cleared between them (its layout key holds n_pad and entries, not the rounded
    slice size), or the shorter call would read the longer call's last chain slots as cell entries."""
    for N, seed in [(1001, 31), (1000, 32), (1001, 33), (1000, 34), (1007, 35), (1000, 31)]:
        check(R, N, 24, 16, 1.0, 0.6, seed, 0)
        assert "realspace_long_kernel" in R.rosen_last_kernel_name()


def test_generation_counter_wrap_of_the_cell_list_kernel(R):
    """As the lattice test of the same name: every warp of the cell-list kernel keeps a generation counter across calls and
    clears its cell table when it wraps (2^19 chains per warp: reachable by a long-lived process). generations_left presets
    the counters so that the wrap falls inside a call, between chains whose entries sit just below the limit."""
    R.rosen_debug_set("realspace_cell_min_n", 2)
    N, n, k, b, sigma, seed = 48, 60000, 8, 1.0, 0.9, 51       # more chains than resident warps: several chains per warp
    s0, t0 = R.rosen_realspace_generate(N, n, k, b, sigma, seed, outputs=("digest", "lnW"))
    assert "realspace_long_kernel" in R.rosen_last_kernel_name()
    o = oracle.realspace_generate(N, 4000, k, b, sigma, seed, outputs=("digest",))
    assert np.array_equal(t0["digest"][:4000].cpu().numpy().view(np.uint64), o.digest)
    import torch
    for left in (0, 1, 3):
        R.rosen_debug_set("generations_left", left)
        s1, t1 = R.rosen_realspace_generate(N, n, k, b, sigma, seed, outputs=("digest", "lnW"))
        assert s1 == s0, left
        assert torch.equal(t0["digest"], t1["digest"]) and torch.equal(t0["lnW"], t1["lnW"]), left
    s2, _ = R.rosen_realspace_generate(N, n, k, b, sigma, seed, outputs=("digest", "lnW"))
    assert s2 == s0


@pytest.mark.parametrize("cap", [None, "33"])
def test_cell_list_kernel_on_short_chains(R, monkeypatch, cap):
    """The knob realspace_cell_min_n = 2 routes short chains through the cell-list kernel, where the oracle's full scan is
    cheap enough for thousands of chains and every k variant; realspace_cand_cap = 33 makes the candidate buffer
    flush after every round, the path dense configurations take."""
    R.rosen_debug_set("realspace_cell_min_n", 2)
    if cap:
        R.rosen_debug_set("realspace_cand_cap", int(cap))
    for N, n, k, b, sigma, seed in [(2, 50, 5, 1.0, 1.0, 1), (3, 3000, 16, 1.0, 1.0, 3), (16, 2001, 7, 0.7, 1.0, 6),
                                    (64, 4000, 16, 1.0, 1.0, 3), (40, 500, 33, 1.0, 0.0, 8), (25, 300, 65, 1.0, 0.8, 11),
                                    (18, 200, 129, 1.0, 1.0, 12), (12, 100, 255, 1.0, 1.0, 12), (256, 300, 64, 1.0, 0.8, 13),
                                    (300, 100, 16, 0.25, 1.0, 14), (200, 100, 8, 1.0, 0.05, 15)]:
        check(R, N, n, k, b, sigma, seed)
        assert "realspace_long_kernel" in R.rosen_last_kernel_name()
    s0, _ = R.rosen_realspace_generate(64, 30011, 16, 1.0, 1.0, 3)
    s1, _ = R.rosen_realspace_generate(64, 30011, 16, 1.0, 1.0, 3, outputs=ALL)
    R.rosen_debug_set("realspace_cell_min_n", 0)
    s2, _ = R.rosen_realspace_generate(64, 30011, 16, 1.0, 1.0, 3)
    assert "realspace_kernel" in R.rosen_last_kernel_name()
    for key in s0:
        if not key.startswith("digest"):
            assert s0[key] == s1[key], key
            assert s0[key] == s2[key] or math.isclose(s0[key], s2[key], rel_tol=1e-12), key


def test_summary_only_variant_bit_identical(R):
    N, n, k = 32, 20011, 16
    s0, _ = R.rosen_realspace_generate(N, n, k, 1.0, 1.0, 3)
    s1, _ = R.rosen_realspace_generate(N, n, k, 1.0, 1.0, 3)
    assert s0 == s1
    s2, _ = R.rosen_realspace_generate(N, n, k, 1.0, 1.0, 3, outputs=ALL)
    for key in s0:
        if not key.startswith("digest"):
            assert s0[key] == s2[key], key


def test_dump_entry_point_and_host_outputs(R):
    N, n, k = 48, 3000, 16
    s, t = R.rosen_realspace_generate(N, n, k, 1.0, 0.8, 13, outputs=("conf", "lnW"))
    s2, conf, lnW = R.rosen_realspace_dump(N, n, k, 1.0, 0.8, 13)
    assert np.array_equal(conf.cpu().numpy(), t["conf"].cpu().numpy())
    assert np.array_equal(lnW.cpu().numpy(), t["lnW"].cpu().numpy())
    s3, th = R.rosen_realspace_generate(N, n, k, 1.0, 0.8, 13, outputs=("conf", "lnW"), host_outputs=True)
    assert np.array_equal(th["conf"].numpy(), t["conf"].cpu().numpy())
    assert s == s3


def test_error_codes(R):
    bad = [((1, 10, 4, 1.0, 1.0, 0), R.ROSEN_EINVAL), ((8, 10, 0, 1.0, 1.0, 0), R.ROSEN_EINVAL),
           ((8, 10, 256, 1.0, 1.0, 0), R.ROSEN_EINVAL), ((8, 10, 4, 0.0, 1.0, 0), R.ROSEN_EINVAL),
           ((8, 10, 4, 1.0, -1.0, 0), R.ROSEN_EINVAL), ((8, 10, 4, float("nan"), 1.0, 0), R.ROSEN_EINVAL),
           ((16384, 10, 4, 1.0, 1.0, 0), R.ROSEN_ERANGE)]
    for args, code in bad:
        with pytest.raises(R.RosenError) as e:
            R.rosen_realspace_generate(*args)
        assert e.value.code == code


def test_config3_full_size_sampled(R):
    """Config 3 at full size (2^22 chains) in the bench launch configuration; sampled chains are
    re-generated one by one by the oracle; physics sanity on the ensemble."""
    w = workloads.CONFIG_3
    s_bench, _ = R.rosen_realspace_generate(w.N, w.n_chains, w.k_trials, w.bond_len, w.sigma, w.seed)
    s, t = R.rosen_realspace_generate(w.N, w.n_chains, w.k_trials, w.bond_len, w.sigma, w.seed,
                                      outputs=("lnW", "digest", "ree2", "alive"))
    for key in s_bench:
        if not key.startswith("digest"):
            assert s_bench[key] == s[key], key
    rng = np.random.default_rng(99)
    ids = np.unique(np.concatenate([rng.integers(0, w.n_chains, 600), [0, w.n_chains - 1]]))
    dg = t["digest"].cpu().numpy().view(np.uint64); lw = t["lnW"].cpu().numpy(); re = t["ree2"].cpu().numpy()
    flips = 0
    for i in ids:
        oi = oracle.realspace_generate(w.N, 1, w.k_trials, w.bond_len, w.sigma, w.seed, chain_offset=int(i),
                                       outputs=("lnW", "digest", "ree2"))
        if oi.digest[0] != dg[i]:
            flips += 1
            continue
        assert (np.isneginf(lw[i]) and np.isneginf(oi.lnW[0])) or math.isclose(lw[i], oi.lnW[0], rel_tol=1e-13)
        assert math.isclose(re[i], oi.ree2[0], rel_tol=1e-12, abs_tol=1e-12)
    assert flips == 0
    assert 0.01 < s["attrition"] < 0.03 and 180 < s["mean_ree2"] < 230     # 1.7 %, ~201


def test_direction_map_vs_oracle(R):
    """R1's direction map alone (rosen_direction_eval) against the oracle's, bit for bit: 200 000 random word pairs and
    every octant edge (the two sides execute the same IEEE operations)."""
    import torch
    rng = np.random.default_rng(777)
    wz = rng.integers(0, 2 ** 32, size=200000, dtype=np.uint64)
    wphi = rng.integers(0, 2 ** 32, size=200000, dtype=np.uint64)
    edge_phi = [(((o << 21) | f) << 8) | low for o in range(8) for f in (0, 1, 0x0FFFFF, 0x100000, 0x1FFFFE, 0x1FFFFF)
                for low in (0, 0xFF)]
    edge_z = [0, 0x1FF, 0x200, 0x80000000, 0x7FFFFFFF, 0xFFFFFE00, 0xFFFFFFFF]
    ez, ep = np.meshgrid(np.array(edge_z, dtype=np.uint64), np.array(edge_phi, dtype=np.uint64))
    wz = np.concatenate([wz, ez.ravel()]); wphi = np.concatenate([wphi, ep.ravel()])
    tz = torch.from_numpy(wz.astype(np.uint32).view(np.int32)).cuda()
    tp = torch.from_numpy(wphi.astype(np.uint32).view(np.int32)).cuda()
    got = R.rosen_direction_eval(tz, tp).cpu().numpy()
    want = np.stack([oracle.direction(int(a), int(b)) for a, b in zip(wz, wphi)])
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))


def test_direction_map_exhaustive_z(R):
    """All 2^23 polar values the map can produce, at one azimuth per octant, against IEEE arithmetic done on the host:
    z = (2q+1) 2^-23 - 1 exactly; a = fl32(1 - z^2) (exact in fp64, rounded once = the fma); rho = IEEE sqrt in fp32;
    u = (fl32(rho c), fl32(rho s), z) with (c, s) the oracle's azimuth factors at z = 2^-23... (rho = 1 there up to one
    rounding, see below). Pins the kernel's own square-root sequence (csrc/direction.cuh sqrt_rn_unit) for every argument."""
    import torch
    q = np.arange(1 << 23, dtype=np.uint64)
    wz = (q << 9).astype(np.uint32)
    z64 = (2.0 * q.astype(np.float64) + 1.0) * 2.0 ** -23 - 1.0                 # exact
    a32 = (1.0 - z64 * z64).astype(np.float32)                                   # 1 - z^2 exact in fp64, one rounding
    rho = np.sqrt(a32)                                                           # IEEE correctly rounded fp32 sqrt
    assert rho.dtype == np.float32 and a32.min() > 2.0 ** -23
    tz = torch.from_numpy(wz.view(np.int32)).cuda()
    for oct_ in range(8):
        wphi = ((oct_ << 21) | 0x0ABCDE) << 8
        # azimuth factors (c, s): the oracle at the equator-most z (q = 2^22: z = 2^-23, a = fl32(1 - 2^-46) = 1, rho = 1)
        cs = oracle.direction(1 << 31, wphi)
        assert cs[2] == np.float32(2.0 ** -23)
        tp = torch.full((1 << 23,), wphi if wphi < 2 ** 31 else wphi - 2 ** 32, dtype=torch.int32, device="cuda")
        got = R.rosen_direction_eval(tz, tp).cpu().numpy()
        ux = (rho.astype(np.float64) * float(cs[0])).astype(np.float32)          # 24 x 24 bit product exact in fp64
        uy = (rho.astype(np.float64) * float(cs[1])).astype(np.float32)
        assert np.array_equal(got[:, 2], z64.astype(np.float32))
        assert np.array_equal(got[:, 0].view(np.uint32), ux.view(np.uint32))
        assert np.array_equal(got[:, 1].view(np.uint32), uy.view(np.uint32))


def test_host_conf_streamed_out_while_the_kernel_runs(R):
    """ROSEN_MEM_HOST + conf with >= 64 virtual blocks: finished chain ranges are copied device -> host on a second stream
    while the kernel still runs. Same bits as the device-buffer call, ragged last virtual block included."""
    N, n, k = 24, 70001, 16
    s_d, t_d = R.rosen_realspace_generate(N, n, k, 1.0, 0.9, 31, outputs=("conf", "lnW", "digest"))
    for _ in range(2):
        s_h, t_h = R.rosen_realspace_generate(N, n, k, 1.0, 0.9, 31, outputs=("conf", "lnW", "digest"), host_outputs=True)
        assert s_h == s_d
        for key in ("conf", "lnW", "digest"):
            assert not t_h[key].is_cuda
            assert np.array_equal(t_h[key].numpy(), t_d[key].cpu().numpy()), key
    o = oracle.realspace_generate(N, 64, k, 1.0, 0.9, 31, chain_offset=n - 64, outputs=("conf",))
    assert np.array_equal(t_h["conf"].numpy()[n - 64:], o.conf)

"""GPU parity of rosen_lattice_perm vs the PERM oracle, tour by tour: digest of all
decisions (growth, enrichment, pruning) bit-exact, flags exact, ln S within 1e-12, weighted means 1e-12."""
import math

import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu
OUT = ("lnW", "alive", "digest", "ree2", "rg2")
INF = float("inf")


@pytest.fixture(scope="module")
def R():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1704_04381_b200 as R
    R.load_library()
    return R


def asymptotic_thresholds(N, lo, hi):
    n = np.arange(N + 1, dtype=np.float64) - 1.0
    ln_c = np.where(n >= 1, math.log(1.21) + n * math.log(4.684) + 0.157 * np.log(np.maximum(n, 1.0)), 0.0)
    return ln_c + math.log(lo), ln_c + math.log(hi), float(ln_c[N])


def compare(R, N, n_tours, seed, ln_lo, ln_hi, ln_ref, max_nodes=1 << 20, offset=0):
    s, t = R.rosen_lattice_perm(N, n_tours, seed, ln_lo, ln_hi, ln_ref, max_nodes=max_nodes, tour_offset=offset, outputs=OUT)
    assert R.rosen_last_kernel_name() == "lattice_perm_kernel"
    o = oracle.lattice_perm(N, n_tours, seed, ln_lo, ln_hi, ln_ref, max_nodes=max_nodes, tour_offset=offset)
    assert np.array_equal(t["digest"].cpu().numpy().view(np.uint64), o.digest)
    assert np.array_equal(t["alive"].cpu().numpy(), o.alive)
    lw = t["lnW"].cpu().numpy()
    have = o.alive != 0
    have &= np.isfinite(o.lnW)
    assert np.array_equal(np.isneginf(lw), np.isneginf(o.lnW))
    assert np.allclose(lw[have], o.lnW[have], rtol=1e-12, atol=1e-12)
    assert np.allclose(t["ree2"].cpu().numpy(), o.ree2, rtol=1e-12, atol=0) and np.allclose(t["rg2"].cpu().numpy(), o.rg2, rtol=1e-12, atol=0)
    for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
        assert s[key] == o.summary[key], key
    for key in ("sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "ln_mean_W"):
        assert math.isclose(s[key], o.summary[key], rel_tol=1e-11), (key, s[key], o.summary[key])
    return s, o


@pytest.mark.parametrize("N,n_tours,lo,hi", [(2, 100, 0.5, 2.0), (3, 500, 0.5, 2.0), (16, 3000, 0.5, 2.0), (33, 2000, 0.9, 1.1),
                                             (64, 1500, 0.3, 3.0), (100, 600, 0.5, 2.0), (257, 100, 0.5, 2.0), (512, 24, 0.5, 2.0)])
def test_perm_parity(R, N, n_tours, lo, hi):
    ln_lo, ln_hi, ln_ref = asymptotic_thresholds(N, lo, hi)
    compare(R, N, n_tours, 5, ln_lo, ln_hi, ln_ref, offset=(1 << 32) - 7)


def test_perm_without_control_is_the_lattice_call(R):
    N = 48
    lo, hi = np.full(N + 1, -INF), np.full(N + 1, INF)
    s, t = R.rosen_lattice_perm(N, 20000, 7, lo, hi, 70.0, outputs=OUT)
    s0, t0 = R.rosen_lattice_generate(N, 20000, 7, outputs=("digest", "lnW", "ree2", "rg2", "alive"))
    assert np.array_equal(t["digest"].cpu().numpy(), t0["digest"].cpu().numpy())
    assert np.array_equal(t["alive"].cpu().numpy(), t0["alive"].cpu().numpy())
    assert s["n_steps_attempted"] == s0["n_steps_attempted"] and s["n_dead"] == s0["n_dead"]
    assert math.isclose(s["mean_ree2"], s0["mean_ree2"], rel_tol=1e-12) and math.isclose(s["ln_mean_W"], s0["ln_mean_W"], rel_tol=1e-12)


def test_perm_node_cap_and_forced_cases(R):
    N = 16
    _, _, ln_ref = asymptotic_thresholds(N, 0.5, 2.0)
    compare(R, N, 64, 2, np.full(N + 1, -INF), np.full(N + 1, -INF), ln_ref, max_nodes=2000)        # enrichment at every step: all capped
    lo = np.full(4, -INF); hi = np.full(4, INF); hi[2] = math.log(5.9)
    s, o = compare(R, 3, 500, 3, lo, hi, 0.0)
    assert math.isclose(s["ln_mean_W"], math.log(30.0), rel_tol=1e-13)                          # 2 leaves x 15 = c_2 in every tour


def test_perm_estimates_at_N100(R):
    """Z_N and <Ree2> from PERM agree with plain Rosenbluth sampling of the library within the joint error, at a fraction of
    the relative variance per growth step."""
    N = 100
    ln_lo, ln_hi, ln_ref = asymptotic_thresholds(N, 0.5, 2.0)
    s, t = R.rosen_lattice_perm(N, 1 << 17, 9, ln_lo, ln_hi, ln_ref, outputs=("lnW", "alive"))
    s0, _ = R.rosen_lattice_generate(N, 1 << 20, 9)
    assert int((t["alive"] == 2).sum()) == 0
    rel_p = math.sqrt(s["sum_w2"]) / s["sum_w"]; rel_r = math.sqrt(s0["sum_w2"]) / s0["sum_w"]     # relative s.e. of the mean weight
    assert abs(s["ln_mean_W"] - s0["ln_mean_W"]) < 5 * math.hypot(rel_p, rel_r)
    assert abs(s["mean_ree2"] / s0["mean_ree2"] - 1.0) < 0.03
    assert rel_p ** 2 * s["n_steps_attempted"] < 0.5 * rel_r ** 2 * s0["n_steps_attempted"]


def test_perm_errors(R):
    N = 8
    lo, hi = np.zeros(N + 1), np.ones(N + 1)
    with pytest.raises(R.RosenError) as e:
        R.rosen_lattice_perm(N, 10, 0, lo, hi, 0.0, outputs=("conf",))
    assert e.value.code == R.ROSEN_EINVAL
    with pytest.raises(R.RosenError) as e:
        R.rosen_lattice_perm(513, 10, 0, np.zeros(514), np.ones(514), 0.0)
    assert e.value.code == R.ROSEN_ERANGE

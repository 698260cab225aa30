"""GPU parity of the model calls (other trial sets, Boltzmann-weighted trials):
rosen_lattice_generate_model / rosen_realspace_generate_model through the C ABI vs the oracle, element by element.
Bars as for the base paths: lattice decisions, trajectory, m sequence bit-exact, sums 1e-12; real space decisions and
coordinates identical bits (flip fraction 0), sums 1e-6."""
import math

import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

ALL = ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")
SUMS = ("sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "ln_mean_W")


@pytest.fixture(scope="module")
def R():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1704_04381_b200 as R
    R.load_library()
    return R


def compare(s, t, o, rel, rg_rel):
    assert np.array_equal(t["digest"].cpu().numpy().view(np.uint64), o.digest), "decision digest"
    assert np.array_equal(t["conf"].cpu().numpy().view(np.uint32), o.conf.view(np.uint32)), "trajectory"
    assert np.array_equal(t["m_seq"].cpu().numpy(), o.m_seq), "m sequence"
    assert np.array_equal(t["alive"].cpu().numpy(), o.alive)
    lnW = t["lnW"].cpu().numpy()
    dead = o.alive == 0
    assert np.all(np.isneginf(lnW[dead])) and np.allclose(lnW[~dead], o.lnW[~dead], rtol=1e-13, atol=0)
    assert np.allclose(t["ree2"].cpu().numpy(), o.ree2, rtol=1e-12, atol=0)
    assert np.allclose(t["rg2"].cpu().numpy(), o.rg2, rtol=rg_rel, atol=0)
    for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
        assert s[key] == o.summary[key], key
    assert math.isclose(s["ln_shift"], o.summary["ln_shift"], rel_tol=1e-13, abs_tol=1e-13)
    for key in SUMS:
        both_nan = math.isnan(s[key]) and math.isnan(o.summary[key])
        assert both_nan or math.isclose(s[key], o.summary[key], rel_tol=rel), (key, s[key], o.summary[key])


@pytest.mark.parametrize("z,beta", [(6, 0.0), (6, 0.3), (6, 0.85), (26, 0.0), (26, 0.25), (26, 0.85)])
@pytest.mark.parametrize("N,n", [(2, 300), (3, 1000), (17, 3001), (64, 2500), (100, 700), (256, 130)])
def test_lattice_model_parity(R, z, beta, N, n):
    s, t = R.rosen_lattice_generate_model(N, n, 21, z=z, beta_eps=beta, chain_offset=(1 << 33) - 5, outputs=ALL)
    assert R.rosen_last_kernel_name().startswith(f"lattice_model_kernel<z={z}")
    o = oracle.lattice_model_generate(N, n, 21, z=z, beta_eps=beta, chain_offset=(1 << 33) - 5)
    compare(s, t, o, 1e-12, 1e-12)


def test_lattice_model_beta0_equals_base_call(R):
    for N in (16, 64, 128):
        s0, t0 = R.rosen_lattice_generate(N, 20000, 7, outputs=("digest", "lnW"))
        s1, t1 = R.rosen_lattice_generate_model(N, 20000, 7, z=6, beta_eps=0.0, outputs=("digest", "lnW"))
        assert np.array_equal(t0["digest"].cpu().numpy(), t1["digest"].cpu().numpy())
        assert s0["digest_xor"] == s1["digest_xor"] and s0["n_dead"] == s1["n_dead"]
        assert math.isclose(s0["mean_ree2"], s1["mean_ree2"], rel_tol=1e-12)
        assert math.isclose(s0["ln_mean_W"], s1["ln_mean_W"], rel_tol=1e-12)


def test_lattice_model_summary_only_and_host_outputs(R):
    s_all, t = R.rosen_lattice_generate_model(48, 5000, 3, z=26, beta_eps=0.4, outputs=ALL)
    s_none, _ = R.rosen_lattice_generate_model(48, 5000, 3, z=26, beta_eps=0.4)
    for key in s_all:
        if not key.startswith("digest"):
            assert s_all[key] == s_none[key], key                       # records + fixed tree: bit-identical
    s_h, th = R.rosen_lattice_generate_model(48, 5000, 3, z=26, beta_eps=0.4, outputs=ALL, host_outputs=True)
    for key in ALL:
        assert np.array_equal(th[key].numpy(), t[key].cpu().numpy()), key


def test_lattice_model_errors(R):
    for args, kw, code in [((1, 10, 0), dict(z=6), R.ROSEN_EINVAL), ((8, 10, 0), dict(z=7), R.ROSEN_EINVAL),
                           ((8, 10, 0), dict(z=6, beta_eps=0.9), R.ROSEN_EINVAL), ((8, 10, 0), dict(z=6, beta_eps=-0.1), R.ROSEN_EINVAL),
                           ((257, 10, 0), dict(z=26), R.ROSEN_ERANGE)]:
        with pytest.raises(R.RosenError) as e:
            R.rosen_lattice_generate_model(*args, **kw)
        assert e.value.code == code


@pytest.mark.parametrize("N,n,k,b,sigma,lam,beta", [
    (2, 100, 4, 1.0, 1.0, 1.5, 0.5), (3, 1000, 16, 1.0, 1.0, 1.5, 0.6), (24, 1500, 16, 1.0, 1.0, 1.5, 0.4),
    (64, 1200, 16, 1.0, 1.0, 1.3, 0.85), (40, 600, 5, 1.0, 0.9, 2.0, 0.3), (33, 500, 1, 1.0, 0.5, 1.5, 0.5),
    (100, 300, 64, 1.0, 0.8, 1.5, 0.4), (50, 300, 255, 1.0, 0.8, 1.25, 0.2), (70, 200, 100, 1.2, 1.0, 1.5, 0.0),
    (300, 40, 64, 1.0, 0.8, 1.5, 0.3)])
def test_realspace_model_parity(R, N, n, k, b, sigma, lam, beta):
    s, t = R.rosen_realspace_generate_model(N, n, k, b, sigma, lam, beta, 17, chain_offset=12345, outputs=ALL)
    o = oracle.realspace_model_generate(N, n, k, b, sigma, lam, beta, 17, chain_offset=12345)
    flips = float((t["digest"].cpu().numpy().view(np.uint64) != o.digest).mean())
    assert flips == 0.0, flips
    compare(s, t, o, 1e-6, 1e-9)


def test_realspace_model_beta0_equals_base_call(R):
    s0, t0 = R.rosen_realspace_generate(64, 8192, 16, 1.0, 1.0, 3, outputs=("digest", "conf"))
    s1, t1 = R.rosen_realspace_generate_model(64, 8192, 16, 1.0, 1.0, 1.5, 0.0, 3, outputs=("digest", "conf"))
    assert np.array_equal(t0["digest"].cpu().numpy(), t1["digest"].cpu().numpy())
    assert np.array_equal(t0["conf"].cpu().numpy(), t1["conf"].cpu().numpy())
    assert math.isclose(s0["mean_ree2"], s1["mean_ree2"], rel_tol=1e-9) and math.isclose(s0["ln_mean_W"], s1["ln_mean_W"], rel_tol=1e-12)


def test_realspace_model_errors(R):
    for args, code in [((8, 10, 4, 1.0, 1.0, 0.9, 0.1, 0), R.ROSEN_EINVAL), ((8, 10, 4, 1.0, 1.0, 1.5, 0.9, 0), R.ROSEN_EINVAL),
                       ((400, 10, 4, 1.0, 1.0, 1.5, 0.1, 0), R.ROSEN_ERANGE)]:
        with pytest.raises(R.RosenError) as e:
            R.rosen_realspace_generate_model(*args)
        assert e.value.code == code


def test_collapse_with_attraction(R):
    """Physics sanity (theta-polymer behaviour): attraction shrinks the chain."""
    r = [R.rosen_lattice_generate_model(48, 1 << 17, 5, z=6, beta_eps=b)[0]["mean_rg2"] for b in (0.0, 0.3, 0.6)]
    assert r[0] > r[1] > r[2]
    r = [R.rosen_realspace_generate_model(32, 1 << 15, 16, 1.0, 1.0, 1.5, b, 5)[0]["mean_rg2"] for b in (0.0, 0.4, 0.8)]
    assert r[0] > r[1] > r[2]

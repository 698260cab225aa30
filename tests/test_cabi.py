"""CPU checks of the boundary: librosen.so loads, exports every symbol include/rosen.h declares, the
pure-host entry points work, and the generate calls fail loudly (no CPU fallback) without a device."""
import ctypes
import math
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def R():
    import paper_1704_04381_b200 as R
    from paper_1704_04381_b200 import build
    build.build()
    R.load_library()
    return R


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rosen.h")).read()
    return sorted(set(re.findall(r"ROSEN_API[^;]*?\b(rosen_\w+)\s*\(", text, flags=re.S)))


def test_every_declared_symbol_is_exported(R):
    from paper_1704_04381_b200 import binding
    names = declared_symbols()
    assert len(names) == 22 and "rosen_lattice_generate" in names and "rosen_realspace_dump" in names
    lib = ctypes.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
        assert hasattr(R, n), f"python binding lacks {n}"


def test_struct_layout_matches_header(R):
    from paper_1704_04381_b200 import binding
    assert ctypes.sizeof(binding.rosen_summary) == 112 == R.SUMMARY_BYTES
    assert ctypes.sizeof(binding.rosen_outputs) == 7 * 8 + 8


def test_host_only_entry_points(R):
    assert "sm_100a" in R.rosen_version()
    assert R.rosen_strerror(R.ROSEN_OK) == "success" and "invalid" in R.rosen_strerror(R.ROSEN_EINVAL)
    assert R.rosen_workspace_bytes() >= 8192 * 64
    assert R.rosen_workspace_release() == R.ROSEN_OK      # nothing allocated yet: still OK
    a = dict(n_chains=10, n_dead=1, n_steps_attempted=90, ln_shift=2.0, sum_w=4.0, sum_w_ree2=8.0, sum_w_rg2=2.0,
             sum_w2=3.0, mean_ree2=2.0, mean_rg2=0.5, attrition=0.1, ln_mean_W=0.0, digest_xor=5, digest_sum=7)
    b = dict(a, n_chains=30, n_dead=0, sum_w=12.0, sum_w_ree2=12.0, digest_xor=6, digest_sum=2 ** 64 - 3)
    m = R.rosen_summary_merge([a, b])
    assert m["n_chains"] == 40 and m["n_dead"] == 1 and m["sum_w"] == 16.0 and m["mean_ree2"] == 20.0 / 16.0
    assert m["digest_xor"] == 3 and m["digest_sum"] == 4 and m["attrition"] == 1 / 40
    # different shifts (long chains, reading A18): rescaled to the largest, exp(2 - 3) on the sums of the first part
    m = R.rosen_summary_merge([a, dict(b, ln_shift=3.0)])
    f = math.exp(-1.0)
    assert m["ln_shift"] == 3.0 and math.isclose(m["sum_w"], 4.0 * f + 12.0, rel_tol=1e-15)
    assert math.isclose(m["sum_w2"], 3.0 * f * f + 3.0, rel_tol=1e-15)
    assert math.isclose(m["ln_mean_W"], 3.0 + math.log((4.0 * f + 12.0) / 40), rel_tol=1e-15)
    with pytest.raises(R.RosenError):
        R.rosen_summary_merge([a, dict(b, ln_shift=float("inf"))])


def test_debug_knobs_validate_and_ignore_the_environment(R, monkeypatch):
    """The knobs exist only behind rosen_debug_set; names and ranges are checked; nothing in the library reads getenv."""
    for knob, good, bad in [("lattice_hash_min_n", 2, 514), ("realspace_cell_min_n", 2049, 1), ("realspace_cand_cap", 33, 32),
                            ("hash_blocks_per_sm", 1, 33)]:
        R.rosen_debug_set(knob, good)
        with pytest.raises(R.RosenError):
            R.rosen_debug_set(knob, bad)
        R.rosen_debug_set(knob, 0)
    with pytest.raises(R.RosenError):
        R.rosen_debug_set("no_such_knob", 1)
    for src in os.listdir(os.path.join(ROOT, "paper_1704_04381_b200", "csrc")):
        if not src.endswith((".cu", ".cuh")):
            continue
        assert "getenv" not in open(os.path.join(ROOT, "paper_1704_04381_b200", "csrc", src)).read(), src


def test_no_cpu_fallback(R):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    lib = R.load_library()
    from paper_1704_04381_b200 import binding
    summ = binding.rosen_summary()
    rc = lib.rosen_lattice_generate(16, 64, 1, 0, None, ctypes.byref(summ), None)
    assert rc == R.ROSEN_ECUDA and R.rosen_last_error() != ""
    rc = lib.rosen_realspace_generate(16, 64, 8, 1.0, 1.0, 1, 0, None, ctypes.byref(summ), None)
    assert rc == R.ROSEN_ECUDA
    assert lib.rosen_lattice_generate(1, 64, 1, 0, None, ctypes.byref(summ), None) == R.ROSEN_EINVAL
    # the round-2 entry points: model calls, PERM, direction map, store probe -- no CPU path either
    assert lib.rosen_lattice_generate_model(16, 64, 1, 0, 26, 0.3, None, ctypes.byref(summ), None) == R.ROSEN_ECUDA
    assert lib.rosen_lattice_generate_noalloc(16, 64, 1, 0, None, None, None) == R.ROSEN_ECUDA
    assert lib.rosen_realspace_generate_model(16, 64, 8, 1.0, 1.0, 1.5, 0.3, 1, 0, None, ctypes.byref(summ), None) == R.ROSEN_ECUDA
    thr = (ctypes.c_double * 17)(*([0.0] * 17))
    assert lib.rosen_lattice_perm(16, 64, 1, 0, thr, thr, 0.0, 1000, None, ctypes.byref(summ), None) == R.ROSEN_ECUDA
    w = (ctypes.c_uint32 * 4)(1, 2, 3, 4)
    out = (ctypes.c_float * 12)()
    assert lib.rosen_direction_eval(w, w, 4, out, R.ROSEN_MEM_HOST, None) == R.ROSEN_ECUDA
    assert lib.rosen_realspace_dump_probe(16, 4, out, None, None) == R.ROSEN_ECUDA


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1704_04381_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "rosen_oracle" not in text, f

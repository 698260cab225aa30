"""rosen_lattice_generate_noalloc against the regular lattice path.

Some programs cannot let a library allocate GPU memory: their own allocator took the whole device at start-up, or their
memory footprint is fixed and audited, or they run a loop that cannot absorb the device-wide stall of cudaMalloc /
cudaFree. For them include/rosen.h has one entry point whose kernel scratch (block partials + the virtual-block ticket)
lives in a static __device__ array inside librosen.so instead of in memory allocated on first use. This file checks that
the entry point

  * gives the same per-chain outputs and the same summary as the existing path (rosen_lattice_generate_async): bit for
    bit below ROSEN_LATTICE_HASH_MIN_N, where both run the same kernel over the same partition -- the bar the lattice
    parity tests use for integer work, and 1e-12 relative (their REL) where the regular call switches kernels;
  * does so on two calls in a row that share the static array (a large call first, then a smaller one with another seed:
    stale partials or a stale ticket from the first call would corrupt the second);
  * leaves the amount of free device memory untouched;
  * refuses sizes beyond its stated maximum with ROSEN_ERANGE and a message that names the limit.

The file name sorts last on purpose: pytest -x stops at the first failure, and this test of an add-on must not hide the
parity tests of the method itself. Within the GPU test the no-allocation calls come FIRST, so that in a fresh process
(pytest tests/test_zz_no_alloc.py) they are the library's very first CUDA work -- the once-per-device set-up path -- while
after the rest of the suite they run on a device the other entry points have long initialised. Both must pass.
"""
import ctypes
import math

import pytest

REL = 1e-12
PER_CHAIN = ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")
INTEGER_FIELDS = ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum")
FLOAT_FIELDS = ("ln_shift", "sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "attrition", "ln_mean_W")


@pytest.fixture(scope="module")
def R():
    import paper_1704_04381_b200 as R
    from paper_1704_04381_b200 import build
    build.build()
    R.load_library()
    return R


def make_outputs(torch, N, n_chains):
    dev = torch.device("cuda", torch.cuda.current_device())
    return {
        "lnW": torch.empty(n_chains, dtype=torch.float64, device=dev),
        "alive": torch.empty(n_chains, dtype=torch.uint8, device=dev),
        "m_seq": torch.empty((n_chains, N - 1), dtype=torch.uint8, device=dev),
        "digest": torch.empty(n_chains, dtype=torch.int64, device=dev),
        "conf": torch.empty((n_chains, N, 3), dtype=torch.int32, device=dev),
        "ree2": torch.empty(n_chains, dtype=torch.float64, device=dev),
        "rg2": torch.empty(n_chains, dtype=torch.float64, device=dev),
    }


def same_bits(torch, a, b):
    """Equality of the stored bits (so that -inf == -inf and a NaN would not slip through as 'not equal')."""
    if a.dtype == torch.float64:
        a, b = a.view(torch.int64), b.view(torch.int64)
    return bool(torch.equal(a, b))


# (N, n_chains, seed, chain_offset, bit_exact). Each row is two calls IN A ROW through the static scratch: the first with
# more virtual blocks than the second, so the second finds the first one's partials and ticket in the array. Sizes span
# several virtual blocks of 2048 chains and a ragged tail; N covers the three scan-kernel variants below the switch-over
# (N % 4 == 0, other N <= 64, 64 < N <= 128) and one length (256) where the regular call uses the hash-map kernel instead.
CASES = [
    ((64, 50_001, 7, 0), (64, 4_097, 8, 12_345), True),
    ((33, 9_001, 3, 1 << 40), (12, 777, 4, 0), True),
    ((100, 6_500, 11, 5), (128, 2_049, 12, 0), True),
    ((256, 5_000, 13, 0), (200, 1_500, 14, 9), False),
]


@pytest.mark.gpu
@pytest.mark.parametrize("first,second,bit_exact", CASES)
def test_noalloc_matches_existing_path_on_two_calls_in_a_row(R, first, second, bit_exact):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    calls = [first, second]
    # everything the caller owns is allocated up front, as such a caller would do
    new_out = [make_outputs(torch, c[0], c[1]) for c in calls]
    new_sum = [torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda") for _ in calls]
    old_out = [make_outputs(torch, c[0], c[1]) for c in calls]
    old_sum = [torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda") for _ in calls]
    for t in new_out:                                  # a call that wrote nothing must not pass by accident
        for v in t.values():
            v.view(torch.uint8).fill_(0xA5)

    # warm-up of exactly these kernel variants (the first launch of a kernel may make the driver load code), then the
    # free-memory reading that the calls under test must leave unchanged
    for (N, n, seed, off), t, s in zip(calls, new_out, new_sum):
        R.rosen_lattice_generate_noalloc(N, n, seed, chain_offset=off, outputs=t, summary_device=s)
    torch.cuda.synchronize()
    for t in new_out:
        for v in t.values():
            v.view(torch.uint8).fill_(0xA5)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()

    # the two calls in a row, same stream, nothing in between
    for (N, n, seed, off), t, s in zip(calls, new_out, new_sum):
        R.rosen_lattice_generate_noalloc(N, n, seed, chain_offset=off, outputs=t, summary_device=s)
        assert R.rosen_last_launch_count() == 2 and "lattice_dp_kernel" in R.rosen_last_kernel_name()
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, f"device memory changed by {free_before - free_after} bytes across no-allocation calls"

    # the existing path on the same inputs
    for (N, n, seed, off), t, s in zip(calls, old_out, old_sum):
        R.rosen_lattice_generate_async(N, n, seed, chain_offset=off, outputs=t, summary_device=s)
    torch.cuda.synchronize()

    for i, (N, n, seed, off) in enumerate(calls):
        tag = f"call {i + 1} (N={N}, n_chains={n})"
        for name in ("alive", "m_seq", "digest", "conf", "ree2"):        # decisions and integers: always bit-exact
            assert same_bits(torch, new_out[i][name], old_out[i][name]), f"{tag}: {name} differs"
        a, b = R.summary_from_device(new_sum[i]), R.summary_from_device(old_sum[i])
        for key in INTEGER_FIELDS:
            assert a[key] == b[key], (tag, key, a[key], b[key])
        assert a["n_chains"] == n
        if bit_exact:
            for name in ("lnW", "rg2"):
                assert same_bits(torch, new_out[i][name], old_out[i][name]), f"{tag}: {name} differs"
            for key in FLOAT_FIELDS:
                assert a[key] == b[key], (tag, key, a[key], b[key])
        else:
            dead = old_out[i]["alive"] == 0
            assert bool(torch.all(torch.isneginf(new_out[i]["lnW"][dead])))
            for name in ("lnW", "rg2"):
                x, y = new_out[i][name][~dead], old_out[i][name][~dead]
                assert bool(torch.all((x - y).abs() <= REL * y.abs())), f"{tag}: {name} beyond {REL}"
            for key in FLOAT_FIELDS:
                assert math.isclose(a[key], b[key], rel_tol=REL, abs_tol=0.0), (tag, key, a[key], b[key])


@pytest.mark.gpu
def test_noalloc_without_outputs_or_summary(R):
    """Both optional arguments left out, then the summary alone: the second call still finds a clean ticket."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    R.rosen_lattice_generate_noalloc(16, 3000, 5)
    s_new = torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda")
    s_old = torch.zeros(R.SUMMARY_BYTES, dtype=torch.uint8, device="cuda")
    R.rosen_lattice_generate_noalloc(16, 3000, 5, summary_device=s_new)
    R.rosen_lattice_generate_async(16, 3000, 5, summary_device=s_old)
    assert R.summary_from_device(s_new) == R.summary_from_device(s_old)


def test_noalloc_rejects_sizes_beyond_the_static_scratch(R):
    """The limits are checked before any CUDA call, so this runs on the CPU box too."""
    from paper_1704_04381_b200 import binding
    assert R.ROSEN_NOALLOC_MAX_N == 512 and R.ROSEN_NOALLOC_MAX_CHAINS == 1 << 24
    assert R.ROSEN_NOALLOC_SCRATCH_BYTES == 8192 * 64 + 256
    lib = ctypes.CDLL(binding.LIB_PATH)
    lib.rosen_lattice_generate_noalloc.argtypes = [ctypes.c_int32, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64,
                                                   ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    assert lib.rosen_lattice_generate_noalloc(R.ROSEN_NOALLOC_MAX_N + 1, 64, 1, 0, None, None, None) == R.ROSEN_ERANGE
    assert "ROSEN_NOALLOC_MAX_N" in R.rosen_last_error()
    assert lib.rosen_lattice_generate_noalloc(64, R.ROSEN_NOALLOC_MAX_CHAINS + 1, 1, 0, None, None, None) == R.ROSEN_ERANGE
    assert "ROSEN_NOALLOC_MAX_CHAINS" in R.rosen_last_error()
    assert lib.rosen_lattice_generate_noalloc(1, 64, 1, 0, None, None, None) == R.ROSEN_EINVAL
    host = binding.rosen_outputs(None, None, None, None, None, None, None, R.ROSEN_MEM_HOST, 0)
    assert lib.rosen_lattice_generate_noalloc(16, 64, 1, 0, ctypes.byref(host), None, None) == R.ROSEN_EINVAL
    assert "device outputs only" in R.rosen_last_error()

"""Memory-safety check without compute-sanitizer (closed on this GPU pool): every per-chain output of every kernel is
written into the middle of a larger sentinel-filled allocation; the guard bands on both sides must come back untouched
and the payload must equal a plain call's. Sizes are ragged (not multiples of the block, group or vector widths)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

ALL = ("lnW", "alive", "m_seq", "digest", "conf", "ree2", "rg2")
GUARD = 4096        # bytes on each side


@pytest.fixture(scope="module")
def R():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1704_04381_b200 as R
    R.load_library()
    return R


def guarded(ref):
    """{name: (raw uint8 buffer, view with ref's shape/dtype inside it)} for the tensors of a reference call."""
    import torch
    out = {}
    for k, t in ref.items():
        nbytes = t.numel() * t.element_size()
        raw = torch.full((GUARD + nbytes + GUARD,), 0xA5, dtype=torch.uint8, device=t.device)
        out[k] = (raw, raw[GUARD:GUARD + nbytes].view(t.dtype).view(t.shape))
    return out


def check_guards(g, ref):
    import torch
    for k, (raw, view) in g.items():
        nbytes = view.numel() * view.element_size()
        assert bool((raw[:GUARD] == 0xA5).all()), f"{k}: write below the buffer"
        assert bool((raw[GUARD + nbytes:] == 0xA5).all()), f"{k}: write above the buffer"
        assert torch.equal(view.view(torch.uint8), ref[k].view(torch.uint8)), f"{k}: payload differs from the plain call"


@pytest.mark.parametrize("N,n", [(2, 1), (7, 333), (64, 1001), (65, 257), (192, 130), (193, 130), (600, 77), (2500, 9)])
def test_lattice_outputs_stay_inside_their_buffers(R, N, n):
    import torch
    _, ref = R.rosen_lattice_generate(N, n, 3, outputs=ALL)
    g = guarded(ref)
    R.rosen_lattice_generate_async(N, n, 3, outputs={k: v for k, (_, v) in g.items()})
    torch.cuda.synchronize()
    check_guards(g, ref)


@pytest.mark.parametrize("N,n,k,sigma", [(2, 1, 1, 1.0), (9, 333, 5, 1.0), (64, 501, 16, 1.0), (33, 100, 255, 0.8),
                                         (256, 37, 64, 0.8), (399, 21, 16, 0.7), (400, 21, 16, 0.7), (3000, 5, 33, 0.3)])
def test_realspace_outputs_stay_inside_their_buffers(R, N, n, k, sigma):
    import torch
    _, ref = R.rosen_realspace_generate(N, n, k, 1.0, sigma, 3, outputs=ALL)
    g = guarded(ref)
    R.rosen_realspace_generate_async(N, n, k, 1.0, sigma, 3, outputs={k_: v for k_, (_, v) in g.items()})
    torch.cuda.synchronize()
    check_guards(g, ref)

"""N > 1 host logic on CPU: world_size-2 gloo ranks shard a chain population by chain_offset
(workloads.shard), each produces its range's summary (here with the oracle, the CPU stand-in for a rank's
GPU), rank 0 gathers and merges them with rosen_summary_merge in rank order. The merged result must equal the
single-range result: counts and digests exactly, sums to 1e-12. No data-path collective exists."""
import math
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, n_total, seed, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import oracle
    import paper_1704_04381_b200 as R
    from paper_1704_04381_b200 import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    offset, count = workloads.shard(n_total, rank, world)
    part = oracle.lattice_generate(N, count, seed, chain_offset=offset, outputs=()).summary
    parts = [None] * world
    dist.all_gather_object(parts, dict(part))
    dist.barrier()
    if rank == 0:
        out.put(R.rosen_summary_merge(parts))
    dist.destroy_process_group()


def test_shard_ranges_cover_population():
    from paper_1704_04381_b200 import workloads
    for n, w in [(10, 3), (1 << 16, 2), (7, 8), (1000, 7)]:
        spans = [workloads.shard(n, r, w) for r in range(w)]
        assert spans[0][0] == 0 and sum(c for _, c in spans) == n
        for (o1, c1), (o2, _) in zip(spans, spans[1:]):
            assert o1 + c1 == o2


@pytest.mark.parametrize("N,n_total,seed", [(16, 4001, 5), (700, 301, 9)])
def test_two_rank_gloo_merge_equals_single_range(N, n_total, seed):
    """(16, ...): equal fixed shifts. (700, ...): a long chain length, where every rank's shift is the largest lnW of its
    own range (reading A18) and rosen_summary_merge rescales the parts to the larger one."""
    import torch.multiprocessing as mp
    import oracle
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, N, n_total, seed, out)) for r in range(2)]
    for p in procs:
        p.start()
    merged = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    whole = oracle.lattice_generate(N, n_total, seed, outputs=()).summary
    for key in ("n_chains", "n_dead", "n_steps_attempted", "digest_xor", "digest_sum"):
        assert merged[key] == whole[key], key
    for key in ("ln_shift", "sum_w", "sum_w_ree2", "sum_w_rg2", "sum_w2", "mean_ree2", "mean_rg2", "ln_mean_W"):
        assert math.isclose(merged[key], whole[key], rel_tol=1e-12), key

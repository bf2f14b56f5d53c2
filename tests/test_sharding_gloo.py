"""The multi-GPU path is z-sharding with no data-path collective; what the ranks share is the
max-over-ranks timing reduction and the rank -> shard mapping of bench.py.  Covered here on CPU with gloo, world 2."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    case = bench.rank_case(1, rank)
    # each rank owns a full-size, distinct shard
    z0 = float(case.z_um[0])
    t = torch.tensor([10.0 + rank], dtype=torch.float64)      # pretend per-rank total ms
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    allz = [None] * world
    dist.all_gather_object(allz, z0)
    q.put((rank, case.n_planes, float(t.item()), allz))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_and_max_timing():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [16, 16]                       # weak scaling: same work per rank
    assert all(abs(r[2] - 11.0) < 1e-12 for r in res)            # MAX over ranks
    assert abs(res[0][3][1] - res[0][3][0] - 0.010) < 1e-12      # distinct z shards


def test_folded_flop_count_matches_survey_formula():
    import bench
    import psf_workloads as W
    for cfg, C in ((1, 3), (3, 3), (5, 5)):
        case = W.get_config(cfg)
        f1, f2 = bench.folded_flops(case)
        N, M, Z = case.pupil_n, case.out_m, case.n_planes
        # 8 N M (N+M) C Z real flop unfolded; even/odd folding cuts it 4x
        assert abs((f1 + f2) - 8.0 * N * M * (N + M) * C * Z / 4.0) < 1e-6 * (f1 + f2)

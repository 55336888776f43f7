"""`-m "not gpu"`: the N > 1 host logic of bench.py with two gloo ranks on the CPU.  The chemistry step has no
inter-cell dependency, so ranks only shard cells ("replicas only"); what needs testing is the
whole-job aggregation (time = MAX over ranks, cells = SUM over ranks) and that every rank draws its own cells."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        from paper_2402_18858_b200 import inputs as I
        ms_local = 10.0 + 5.0 * rank          # rank 1 is the slow one
        cells_local = 1000 * (rank + 1)
        ms, cells = bench.aggregate_over_ranks(ms_local, cells_local, dist, torch.device("cpu"))
        cfg = I.get_config("c0")
        prob = I.make_problem(cfg, n=256, seed=cfg.index + 1000 * rank)  # the seeding rule of bench.run_ours
        t = torch.tensor([float(prob.state.T[:8].sum())], dtype=torch.float64)
        gathered = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(gathered, t)
        if rank == 0:
            out.put((ms, cells, [float(g.item()) for g in gathered]))
    finally:
        dist.destroy_process_group()


def test_two_rank_aggregation_and_sharding():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    ms, cells, sums = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 15.0            # MAX over ranks
    assert cells == 3000         # SUM over ranks
    assert sums[0] != sums[1]    # every rank owns its own seeded cells (weak scaling, no shared data)


def test_single_rank_aggregation_is_identity():
    import bench
    assert bench.aggregate_over_ranks(3.5, 42, None, None) == (3.5, 42)


def test_roofline_traffic_comes_from_the_tracked_ncu_table():
    """bench.py's roofline.traffic is read from profiles/ncu_dram_bytes.csv (ncu --set full captures), never a literal in
    the code; a configuration without a capture yields None, and so does a capture taken from other kernel sources than
    this tree's (each row names the csrc_sha() it was measured on)."""
    import bench
    cap = bench.dram_capture_from_profiles("bf16_fused", 2, 1048576)
    assert cap is not None and 1.5e9 < cap["bytes"] < 2.0e9   # state in + h2 out of the fused kernel at configs[2]
    assert cap["source"].startswith("profiles/") and len(cap["csrc_sha"]) == 16
    sha = bench.csrc_sha()
    assert len(sha) == 16 and int(sha, 16) >= 0
    # a capture of these sources is reported, one of other sources is not
    assert bench.dram_bytes_from_profiles("bf16_fused", 2, 1048576, sha=cap["csrc_sha"]) == cap["bytes"]
    assert bench.dram_bytes_from_profiles("bf16_fused", 2, 1048576, sha="0" * 16) is None
    assert bench.dram_bytes_from_profiles("bf16_fused", 3, 4194304) is None
    assert bench.dram_bytes_from_profiles("bf16_tail", 2, 12345) is None

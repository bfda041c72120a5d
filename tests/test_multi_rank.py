"""N > 1 path of bench.py on CPU: world_size-2 gloo.  Ranks own disjoint contiguous event ranges of the seeded
stream (no data-path collective); only the step time is reduced with MAX."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import rambo as I
from paper_2503_21935_b200.shard import max_over_ranks, rank_range


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, per_rank, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        start, stop = rank_range(per_rank, rank, world)
        mom = I.make_momenta("gg_ttg", stop - start, seed=1, start=start)
        gs = I.make_gs(stop - start, seed=1, alphas=None, start=start)
        # every rank gathers the (start, stop, checksum) triples: ranges must tile the global stream
        mine = torch.tensor([start, stop, float(mom.sum()), float(gs.sum())], dtype=torch.float64)
        allr = [torch.zeros(4, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(allr, mine)
        t = max_over_ranks(1.0 + rank, dist)
        dist.barrier()
        if rank == 0:
            out.put((np.stack([x.numpy() for x in allr]), t))
    finally:
        dist.destroy_process_group()


def test_two_ranks_own_disjoint_ranges_and_reduce_time_with_max():
    world, per_rank = 2, 1000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, per_rank, q)) for r in range(world)]
    for p in procs:
        p.start()
    table, tmax = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert tmax == 2.0  # max over ranks of (1 + rank)
    assert table[0][0] == 0 and table[0][1] == table[1][0] and table[1][1] == world * per_rank
    # the shards are slices of the one global stream (counter-based generator): no overlap, nothing skipped
    full = I.make_momenta("gg_ttg", world * per_rank, seed=1)
    gs = I.make_gs(world * per_rank, seed=1, alphas=None)
    for r in range(world):
        s, e = int(table[r][0]), int(table[r][1])
        assert np.isclose(table[r][2], full[s:e].sum(), rtol=1e-13)
        assert np.isclose(table[r][3], gs[s:e].sum(), rtol=1e-13)


def test_rank_range_errors():
    import pytest
    assert rank_range(10, 3, 4) == (30, 40)
    with pytest.raises(ValueError):
        rank_range(10, 4, 4)


def test_bench_reference_arm_under_a_two_rank_launcher():
    """bench.py's launcher contract on CPU: under torchrun with 2 ranks the reference arm prints ONE JSON line (rank 0)
    and every rank exits 0 (the other rank leaves without work)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--process", "gg_tt", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"


def test_bench_gpus_flag_spawns_its_own_ranks():
    """`python bench.py --gpus 2` without a launcher re-executes itself under torchrun (checked with the reference arm,
    which needs no GPU)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2", "--process", "gg_tt",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2

"""N > 1 path of bench.py on CPU: two `gloo` ranks (world_size 2, 127.0.0.1).  The renderer shards by
independent replicas only (DESIGN.md §5 "replicas only": no data-path collective), so what there is to test is
the host logic: max-over-ranks timing, whole-job throughput, and that --impl reference prints on rank 0 only."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 if rank == 0 else 12.5          # rank 1 is the slow one
    ms_max, value = bench.aggregate_replicas(ms_local, 640 * 480, 100, world, dist, "cpu")
    dist.barrier()
    q.put((rank, ms_max, value))
    dist.destroy_process_group()


def test_replica_aggregation_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    expect = 640 * 480 * 100 * 2 / 12.5e-3 / 1e6     # work of BOTH ranks / slowest rank's time
    for rank, ms_max, value in res:
        assert ms_max == 12.5
        assert abs(value - expect) < 1e-9 * expect


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    ms_max, value = bench.aggregate_replicas(4.0, 1000, 10, 1, None, "cpu")
    assert ms_max == 4.0 and abs(value - 1000 * 10 / 4e-3 / 1e6) < 1e-12


def test_reference_arm_prints_on_rank0_only():
    """bench.py --impl reference (the CPU oracle) under a 2-rank launch: rank 0 prints one JSON line, rank 1 nothing."""
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1",
                            "--gpus", "2", "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
    assert outs[1] == ""

"""N > 1 bookkeeping of bench.py on CPU: two gloo processes (world_size 2).  The path itself has no
exchange step (replicas only), so what has to be right is: disjoint per-rank
chunks, max-over-ranks timing, whole-job aggregation, and that only rank 0 prints the reference line."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank            # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world, device="cpu")
    seeds = bench.rank_chunk_seeds(rank)
    gathered = [None] * world
    dist.all_gather_object(gathered, seeds)
    dist.barrier()
    q.put((rank, ms, gathered, bench.aggregate_value(18336, 100, world, ms)))
    dist.destroy_process_group()


def test_two_rank_bookkeeping_gloo():
    world, port = 2, 29731
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, gathered, value in res:
        assert ms == 15.0                               # max over ranks, on every rank
        assert not set(gathered[0]) & set(gathered[1])  # disjoint chunks per rank (weak scaling)
        assert abs(value - 2 * 18336 * 100 / 15e-3) < 1e-6 * value


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["metric"] == "channel_pair_spectra_per_s"

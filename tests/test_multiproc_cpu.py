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


# --------------------------------------------------------------------------------------------
# f4: strong scaling of ONE shot ("halves with each doubling", L217 "embarrassingly parallel"): the chunks
# of a shot are dealt round-robin to the ranks (bench.py --workload streamed --scaling strong), every rank takes the
# offsets from chunk 0 itself (no broadcast), no collective on the data path.  On CPU the per-chunk analysis is the
# float64 pipeline of oracle/fft_baseline.py (the GPU run of the same split is timed by bench.py; a chunk analysed alone
# and inside a stream give the same bits there: tests/test_parity_gpu.py::test_config4_streamed_shot).
def _shot(n_chunks=6, C=6, T=1200, seed=11):
    import numpy as np
    rng = np.random.default_rng(seed)
    o_true = rng.uniform(2000, 3000, size=C)
    sig = rng.standard_normal((C, n_chunks * T))
    sig[1] += 0.7 * sig[0]
    counts = np.rint(o_true[:, None] + 200 * sig).astype(np.int16)
    return np.stack([counts[:, n * T:(n + 1) * T] for n in range(n_chunks)])


def _analyze_chunk_cpu(counts_n, offs):
    from oracle import delta_oracle as o
    from oracle import fft_baseline as fb
    y = o.normalise(counts_n, offs, o.NORM_RELATIVE)
    return fb.analyze_chunk(y, 128, 64, 64)


def _strong_worker(rank, world, port, q):
    import numpy as np
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    from oracle import delta_oracle as o
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    shot = _shot()
    offs = o.offsets(shot[0][:, :500])                    # every rank: from chunk 0 of the shot
    mine = bench.shot_chunks_of_rank(shot.shape[0], rank, world)
    res = {n: _analyze_chunk_cpu(shot[n], offs) for n in mine}
    digest = {n: {k: float(np.sum(v)) for k, v in r.items()} for n, r in res.items()}
    gathered = [None] * world
    dist.all_gather_object(gathered, (mine, digest))      # bookkeeping only: the data path has no collective
    dist.barrier()
    q.put((rank, gathered, {n: r["G"] for n, r in res.items()}))
    dist.destroy_process_group()


def test_strong_scaling_split_of_one_shot_gloo():
    import numpy as np
    from oracle import delta_oracle as o
    world, port = 2, 29733
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_strong_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=300) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    shot = _shot()
    offs = o.offsets(shot[0][:, :500])
    serial = {n: _analyze_chunk_cpu(shot[n], offs) for n in range(shot.shape[0])}
    seen = []
    for rank, gathered, G_by_chunk in res:
        mine, _ = gathered[rank]
        assert mine == list(range(rank, shot.shape[0], world))           # chunk n -> rank n mod world
        for n, G in G_by_chunk.items():
            assert np.array_equal(G, serial[n]["G"])                     # bit-identical whichever rank ran the chunk
            seen.append(n)
        # every rank sees the same global picture
        all_chunks = sorted(n for m, _ in gathered for n in m)
        assert all_chunks == list(range(shot.shape[0]))                  # every chunk exactly once
        for m, dig in gathered:
            for n in m:
                for k, v in dig[n].items():
                    assert v == float(np.sum(serial[n][k]))
    assert sorted(seen) == list(range(shot.shape[0]))

"""Multi-GPU host logic on CPU: world_size 2, gloo.

Events are independent units: rank r generates / processes events [r*n, (r+1)*n) and the only collectives are the
MAX (time) and SUM (work) of bench.py's scalars.  Run here without a GPU."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import bench
    from workloads import generate_events, get_workload
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n = 3
    w, batch = bench.make_batch(3, n, rank)
    assert list(bench.shard_event_range(rank, n)) == list(range(rank * n, (rank + 1) * n))
    # the rank's shard is bit-identical to the same events generated in one process
    ref = generate_events(get_workload(3).scaled(world * n), events=range(rank * n, (rank + 1) * n))
    assert np.array_equal(batch.hits_xy, ref.hits_xy) and np.array_equal(batch.event_offsets, ref.event_offsets)
    ms, (votes, events, hits) = bench.reduce_job(10.0 + rank, 100.0 * (rank + 1), batch.n_events, batch.n_hits, world, "cpu")
    tot_hits = torch.tensor([float(batch.n_hits)], dtype=torch.float64)
    dist.all_reduce(tot_hits)
    assert ms == 10.0 + (world - 1)                       # MAX over ranks
    assert votes == 100.0 * sum(range(1, world + 1)) and events == world * n and hits == float(tot_hits.item())
    np.save(os.path.join(out_dir, f"hits_{rank}.npy"), batch.hits_xy)
    dist.barrier()
    dist.destroy_process_group()


def test_event_sharding_and_scalar_reduction_world_2(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    a, b = np.load(tmp_path / "hits_0.npy"), np.load(tmp_path / "hits_1.npy")
    assert a.shape[0] > 0 and b.shape[0] > 0 and not (a.shape == b.shape and np.array_equal(a, b))   # disjoint shards


def test_reference_arm_runs_on_rank_0_only(tmp_path):
    """bench.py --impl reference under a 2-rank launch: rank 0 prints the line, rank 1 exits 0 without work."""
    import subprocess
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"; env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    import json
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0

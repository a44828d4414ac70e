"""The N > 1 path of bench.py on CPU (world_size 2, gloo): the path shards by sequence with no data-path collective
("replicas only"), so what there is to check is the host logic -- every rank builds a same-shaped
batch from its own seed, the reported step time is the max over ranks, and only rank 0 of the reference arm works."""
import json
import os
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = bench.rank_workload("mini3", rank)
    step = bench.max_over_ranks(100.0 + 7.0 * rank, torch.device("cpu"), world)
    digest = int(np.bitwise_xor.reduce(wl.sel_k.reshape(-1).astype(np.uint64)))
    gathered = [None] * world
    dist.all_gather_object(gathered, (wl.seed, wl.sel_k.shape, wl.seq_len.tolist(), digest))
    dist.barrier()
    if rank == 0:
        with open(out, "w") as f:
            json.dump({"step": step, "ranks": gathered}, f)
    dist.destroy_process_group()


def test_two_ranks_build_distinct_same_shaped_batches_and_report_the_slowest(tmp_path):
    out = str(tmp_path / "r.json")
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["step"] == 107.0                                   # max over ranks, not rank 0's own 100.0
    (s0, shape0, len0, d0), (s1, shape1, len1, d1) = r["ranks"]
    assert s1 == s0 + 1000 and shape0 == shape1 and len0 == len1
    assert d0 != d1                                             # different sequences, same shapes


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "cfg1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "cfg1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=300)
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["n_gpus"] == 2
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0

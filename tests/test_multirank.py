"""N > 1 path (replicas only): world_size-2 gloo runs on CPU of the only cross-rank
logic there is -- bench.py's measurement aggregation (time = max over ranks, work = sum over ranks) and the
per-rank workload seeding -- plus the reference arm's "rank 0 alone prints" rule."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from workloads import BASE_SEED, CONFIGS, make_workload

    cfg = CONFIGS["c4"].scaled(name="c4_mr", n_carts=12, n_slots=12, B=3, len_mu=5.0, len_min=20, len_max=300,
                               lq_min=30, lq_max=200, n_dist_max=3)
    wl = make_workload(cfg, BASE_SEED + rank)              # bench.py: every rank draws its own batch
    fwd, bwd = bench.attn_flops(wl)
    ms = 3.0 + rank                                        # rank 1 is the slow one
    got = bench.reduce_over_ranks(ms, 10.0 - rank, fwd + bwd, world, "cpu")
    out[rank] = (got, fwd + bwd, int(wl.pairs_per_head()))
    dist.destroy_process_group()


def test_replica_aggregation_gloo_world2():
    world, port = 2, _free_port()
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    (ms0, e0, f0), w0, p0 = res[0]
    (ms1, e1, f1), w1, p1 = res[1]
    assert p0 != p1 and w0 != w1                           # different seeds: different ragged batches
    assert ms0 == ms1 == 4.0                               # max over ranks
    assert e0 == e1 == 10.0
    assert f0 == f1 == w0 + w1                             # sum over ranks


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "c1", "--steps", "1",
           "--warmup", "0", "--gpus", "2"]
    r1 = subprocess.run(cmd, env=dict(env, RANK="1", LOCAL_RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(env, RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and np.isfinite(line["value"]) and line["value"] > 0

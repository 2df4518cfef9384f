"""Multi-GPU host logic on CPU (gloo, world_size 2): the path shards by independent frames -- "replicas only",
DESIGN.md §9 -- so the N > 1 logic is (1) every rank draws its own, disjoint frames of the same code, (2) the
reported time is the max over ranks, (3) the value counts the frames of all ranks, and (4) under --impl reference
rank 0 alone prints."""
import json
import os
import subprocess
import sys

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    sys.path.insert(0, ROOT)
    import bench
    from paper_1702_07740_b200 import workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = W.CONFIGS[1]
    base = W.make_base_matrix(cfg.code)
    seed_base = bench.rank_seed_base(cfg.index, rank)
    fr = W.make_frames(base, cfg.code.Z, W.sigma_for_gap(cfg.code.rate, cfg.gaps_db[0]), 4, seed_base)
    # same code on every rank, different frames
    digest = torch.tensor([float(base.sum()), float(fr.llr.astype(np.float64).sum())], dtype=torch.float64)
    gathered = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(gathered, digest)
    ms_local = 10.0 * (rank + 1)                     # pretend rank 1 is the slow one
    ms = bench.max_over_ranks([ms_local], dist, torch.device("cpu"))[0]
    value = bench.decoded_mbit_per_s(cfg.code.n, 4 * world, ms * 1e-3)
    if rank == 0:
        out.put({"gathered": [g.tolist() for g in gathered], "ms": ms, "value": value})
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_over_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    res = out.get()
    (b0, l0), (b1, l1) = res["gathered"]
    assert b0 == b1 and l0 != l1                     # one code, disjoint frames
    assert res["ms"] == 20.0                         # max over ranks
    assert res["value"] == 2560 * 8 / 20e-3 / 1e6    # frames of ALL ranks / max time


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--config", "1", "--ref-iters", "5"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]

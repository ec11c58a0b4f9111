"""The N > 1 path of bench.py is replicas only: no data-path collective, one bunch per rank.
Its host logic -- per-rank seeds, max-over-ranks timing, whole-job rate, rank 0 alone printing, the reference arm's
idle ranks -- runs here on CPU with world_size 2 over gloo."""
import json
import os
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    from workloads import make_config
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank                              # rank 1 is the slow one
    ms_max = bench.max_over_ranks(ms_local, world, "cpu")
    rate = bench.aggregate_rate(1000, 4, world, ms_max)
    wl = make_config(3, n=64, seed=bench.rank_seed(3, rank))
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms_max": ms_max, "rate": rate, "x0": float(wl.particles["x"][0]), "seed": bench.rank_seed(3, rank)}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_replica_logic_world_size_2_gloo(tmp_path):
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = (json.load(open(tmp_path / f"r{r}.json")) for r in (0, 1))
    assert r0["ms_max"] == r1["ms_max"] == 15.0               # the slowest rank's time, on every rank
    assert r0["rate"] == r1["rate"] == 2 * 1000 * 4 / 15.0e-3  # units of ALL ranks over that time
    assert r0["seed"] is None and r1["seed"] == 1003          # own bunch per rank, rank 0 = the config's seed
    assert r0["x0"] != r1["x0"]


def test_reference_arm_prints_on_rank_0_only():
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29999")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--ref-sample-particles", "500"]
    out1 = subprocess.run(cmd, env=dict(env, RANK="1"), capture_output=True, text=True, timeout=300)
    assert out1.returncode == 0 and out1.stdout.strip() == ""
    out0 = subprocess.run(cmd, env=dict(env, RANK="0"), capture_output=True, text=True, timeout=300)
    assert out0.returncode == 0
    line = json.loads(out0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert np.isclose(line["e2e"]["value"], line["value"])

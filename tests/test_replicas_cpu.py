"""N > 1 host logic of bench.py (replicas only) on CPU: two gloo ranks on 127.0.0.1.
Each rank works on its own layer (different seeds), there is no data-path collective, the job's time is
the MAX over ranks and the value is the units of all ranks over that time; `--impl reference` runs on
rank 0 alone."""
import os
import subprocess
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    import bench
    from paper_2607_01065_b200 import inputs
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_s = 0.010 * (1 + rank)                    # rank 1 is the slow one
    value, max_s = bench.whole_job_value(local_s, 1000.0, world, "cpu")
    seed = bench.rank_seed(1, "k", rank)
    x = inputs.k_like(1, 8, 128, seed)
    gathered = [None] * world
    dist.all_gather_object(gathered, (float(value), float(max_s), int(seed), float(np.abs(x).sum())))
    if rank == 0:
        out.put(gathered)
    dist.destroy_process_group()


def test_two_rank_replica_aggregation():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (v0, m0, s0, a0), (v1, m1, s1, a1) = res
    assert m0 == m1 == 0.020                         # MAX over ranks
    assert v0 == v1 == 2 * 1000.0 / 0.020            # whole-job units over the slowest rank's time
    assert s0 != s1 and a0 != a1                     # independent layers per rank
    from paper_2607_01065_b200 import inputs
    assert s0 == inputs.seed_of(1, "k")             # rank 0 is the documented seed


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` times the oracle on the host cores and prints ONE JSON line with the contract's keys."""
    import json
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "1", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-500:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "KV vectors/s" and d["higher_is_better"] is True
    assert d["config"]["workload"].startswith("cfg4:") and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == dict(value=d["value"], unit=d["unit"], h2d_bytes_per_step=0, d2h_bytes_per_step=0)

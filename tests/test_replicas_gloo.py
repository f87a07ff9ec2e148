"""The N > 1 path of bench.py is "replicas only": no data-path collective, one MAX all-reduce
of the timing scalar.  Its host logic is exercised here with world_size 2 over gloo on the CPU; the labeling itself
is replaced by the oracle (this is a test of the plumbing, not of the kernels)."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    import numpy as np
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    from oracle import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    plan = bench.replica_plan(rank, cfg=4)
    n = 1 << 12
    src, dst, _ = oracle.gen_regular(n, 3, plan["seed"])
    mask, _ = oracle.gen_occupancy(src.size, 0.5, plan["seed"], plan["realization"])
    labels = oracle.label(n, src, dst, mask)
    local_ms = 10.0 * (rank + 1)                                  # rank 1 is the slow one
    total_ms = bench.max_over_ranks(local_ms, world, "cpu")
    dist.barrier()
    with open(os.path.join(out_dir, "rank%d.json" % rank), "w") as f:
        json.dump({"plan": plan, "total_ms": total_ms, "n_clusters": int((labels == np.arange(n)).sum()),
                   "mask_sum": int(mask.sum()), "value": bench.job_value(world, 1, src.size, total_ms)}, f)
    dist.destroy_process_group()


def test_two_replicas_over_gloo(tmp_path):
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0 = json.load(open(tmp_path / "rank0.json"))
    r1 = json.load(open(tmp_path / "rank1.json"))
    assert r0["plan"]["seed"] == r1["plan"]["seed"] and (r0["plan"]["realization"], r1["plan"]["realization"]) == (0, 1)
    assert r0["mask_sum"] != r1["mask_sum"]                       # different realizations: independent replicas
    assert r0["total_ms"] == r1["total_ms"] == 20.0                # max over ranks
    assert abs(r0["value"] - 2 * 6144 / 20e-3 / 1e9) < 1e-12       # all ranks' bonds over the slowest rank's time


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--workload", "cfg1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--workload", "cfg1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2

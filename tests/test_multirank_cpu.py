"""World-size-2 gloo tests (CPU) of bench.py's multi-rank logic.  The path does not shard (north_star:
one GPU, no collectives), so N > 1 means independent replicas: the only cross-rank step is the
max-over-ranks of the device time and the aggregate throughput."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 100.0 if rank == 0 else 250.0               # the slower rank sets the job's time
    tmax, value = bench.aggregate(ms, bodies_per_rank=1000, steps=10, world=world)
    dist.barrier()
    out[rank] = (tmax, value)
    dist.destroy_process_group()


def test_aggregate_max_over_ranks_gloo():
    world, port = 2, 29641
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        tmax, value = res[r]
        assert tmax == 250.0
        assert value == world * 1000 * 10 / 0.250


def test_reference_arm_prints_one_json_line_and_only_on_rank0():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "c1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["dtype"] == "f64" and d["higher_is_better"] is True
    env["RANK"] = "1"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "c1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0 and r.stdout.strip() == ""

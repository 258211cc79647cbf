"""N > 1 bookkeeping of bench.py on CPU (gloo, world_size 2): the path itself does not communicate
("replicas only"); what the ranks share is the max-over-ranks time and the
aggregate throughput."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 20.0 - 3.0 * rank], world, "cpu")
    dist.barrier()
    if rank == 0:
        with open(out, "w") as fh:
            json.dump({"ms": ms, "e2e": e2e, "value": bench.aggregate_value(1000, 4, world, ms)}, fh)
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate(tmp_path):
    out = str(tmp_path / "r.json")
    mp.spawn(_worker, args=(2, 29671, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["ms"] == 15.0 and r["e2e"] == 20.0                 # maxima over the two ranks
    assert r["value"] == 2 * 1000 * 4 / 15.0e-3                 # both replicas' units over the slowest time


def test_reference_arm_is_silent_off_rank_zero():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, env=env, timeout=120)
    assert res.returncode == 0 and res.stdout.strip() == ""


def test_flop_accounting_matches_design():
    sys.path.insert(0, ROOT)
    import bench
    assert abs(bench.flop_per_unit(3, 21, 400) - (264.0 + 10164.0 / 400.0)) < 1e-12
    assert bench.flop_per_unit(2, 5, 41) == 2.0 * 2 * 12 + (2.0 * 2 * 6 * 15 + 8.0 * 15) / 41

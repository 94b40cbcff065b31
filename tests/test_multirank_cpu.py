"""N > 1 plumbing of bench.py on CPU: two gloo ranks, "replicas only".

The data path has no collective; the only cross-rank step is the reduction of the timing
(max over ranks) and of the processed units (sum over ranks), bench.aggregate().
"""
import json
import os
import socket
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (10 + 5 r) ms and processed (100 + r) units
    ms, units = bench.aggregate(10.0 + 5.0 * rank, 100.0 + rank, dist, None)
    dist.barrier()
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "units": units}, f)
    dist.destroy_process_group()


def test_aggregate_max_time_sum_units_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        with open(tmp_path / f"r{r}.json") as f:
            d = json.load(f)
        assert d["ms"] == 15.0              # max over ranks
        assert d["units"] == 201.0          # sum over ranks


def test_aggregate_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.0, 7.0) == (3.0, 7.0)


def test_reference_arm_nonzero_ranks_exit_without_work():
    """Under torchrun only rank 0 runs the oracle; other ranks exit 0 and print nothing."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "2", "--warmup", "3"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""

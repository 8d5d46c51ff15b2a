"""N > 1 path of bench.py on CPU: world_size-2 gloo run of the only cross-rank logic the path has (replicas:
a barrier and the max over ranks of the device time), plus the reference arm's rank rule."""
import json
import os
import socket
import subprocess
import sys

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
    sec = bench.max_over_ranks(0.5 + 0.25 * rank, world, "cpu")      # rank 1 is the slow one
    dist.barrier()
    val = bench.whole_job_value(1000, 4, world, sec)
    with open(os.path.join(out, f"r{rank}.json"), "w") as f:
        json.dump({"sec": sec, "value": val}, f)
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"r{k}.json")) for k in range(2)]
    assert r[0]["sec"] == r[1]["sec"] == 0.75                       # the slowest rank's time, on every rank
    assert r[0]["value"] == 2 * 1000 * 4 / 0.75                     # both replicas' points over that time


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(1.25, 1, "cpu") == 1.25
    assert bench.whole_job_value(10, 3, 1, 2.0) == 15.0


def test_reference_arm_only_rank0_prints(tmp_path):
    """bench.py --impl reference under a 2-rank launch: rank 0 prints one JSON line, rank 1 exits 0 silently."""
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    outs = []
    for rank in (0, 1):
        e = dict(env, RANK=str(rank), LOCAL_RANK=str(rank))
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--config", "0", "--steps", "1", "--warmup", "0", "--fixed-iters", "2"],
                           env=e, capture_output=True, text=True, timeout=300)
        assert p.returncode == 0, p.stderr
        outs.append(p.stdout.strip())
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
    assert outs[1] == ""

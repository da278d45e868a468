"""world_size-2 gloo tests (CPU) of the N > 1 path: replicas only -- each rank times its own solve,
the job time is the max over ranks, rank 0 alone reports; the reference arm runs on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    mine = 10.0 + 5.0 * rank                    # rank 1 is the slow replica
    dist.barrier()
    got = bench.max_over_ranks(mine, world, "cpu")
    out[rank] = got
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    port = _free_port()
    mgr = mp.get_context("spawn").Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0] == 15.0 and out[1] == 15.0


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, WORLD_SIZE="2", OMP_NUM_THREADS="2")
    outs = []
    for rank in (0, 1):
        env["RANK"] = str(rank)
        env["LOCAL_RANK"] = str(rank)
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--config", "1", "--steps", "1", "--warmup", "1"], env=env, capture_output=True,
                           text=True, timeout=300)
        assert p.returncode == 0, p.stderr
        outs.append(p.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["unit"] == "s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0

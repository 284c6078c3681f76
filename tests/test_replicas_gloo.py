"""The N > 1 path is "replicas only": no data-path collective, the ranks meet only in bench.py's barrier
and MAX-over-ranks of the elapsed time.  That host logic is covered here with world_size 2 on CPU (gloo)."""
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
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 * (rank + 1), dist, "cpu")  # rank 0: 10 ms, rank 1: 20 ms
    dist.barrier()
    out[rank] = ms
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2():
    sys.path.insert(0, ROOT)
    import bench

    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
        assert out[0] == out[1] == 20.0
    # two replicas of V sites, 3 sweeps each, slowest took 20 ms
    assert bench.aggregate_value(2, 4096, 3, 20.0) == 2 * 4096 * 3 / 0.020
    assert bench.max_over_ranks(7.5, None, "cpu") == 7.5


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference",
           "--gpus", "2", "--config", "cfg0", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_bench_gpus_n_without_a_launcher_spawns_n_ranks():
    """`python bench.py --gpus 2` with WORLD_SIZE unset must become two ranks itself (missing 2(ii)): the
    command it builds is torchrun's, and run end to end (reference arm: no GPU needed) it prints n_gpus = 2."""
    sys.path.insert(0, ROOT)
    import bench

    cmd = bench.spawn_command(2, ["--gpus", "2", "--steps", "1"], port=29999)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=2" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29999"
    assert cmd[-5] == os.path.join(ROOT, "bench.py") and cmd[-4:] == ["--gpus", "2", "--steps", "1"]
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env["OMP_NUM_THREADS"] = "2"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--config",
                        "cfg0", "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600,
                       cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2

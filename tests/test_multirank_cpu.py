"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): replicas only -- the ranks share
no data; the job time is the max over ranks and the value the sum of the replicas' work.
The reference arm prints on rank 0 only."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, device="cpu")
    dist.barrier()
    q.put((rank, ms, bench.job_value(world, 1e9, ms)))
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]                     # max over ranks on every rank
    assert all(abs(r[2] - 2 * 1e9 / 15e-3 * 1e-9) < 1e-9 for r in res)  # two replicas' work / max time


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, device="cpu") == 3.5
    assert bench.step_flops(10) == 2 * 1320 * 10 + 2 * 504 * 10


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                        "--warmup", "1"], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["metric"] == "wilson_clover_dslash_gflops"


def test_gpus_flag_spawns_one_rank_per_gpu_on_localhost():
    """`bench.py --gpus N` without a launcher starts its own N ranks (it used to run
    one replica and print n_gpus: 1); without N devices it refuses instead of under-reporting."""
    import argparse
    import pytest
    sys.path.insert(0, ROOT)
    import bench
    cmd = bench.replica_command(4, 29511, ["--gpus", "4", "--steps", "7"])
    assert cmd[1:3] == ["-m", "torch.distributed.run"]
    assert "--nproc-per-node" in cmd and cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "7"] and cmd[-5].endswith("bench.py")
    with pytest.raises(SystemExit) as e:
        bench.spawn_replicas(argparse.Namespace(gpus=1024))
    assert "1024" in str(e.value)
